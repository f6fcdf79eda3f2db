// The hot path of liboat.so for sm_100a (B200): the marching kernels of H (projection, steps A2-A4 of
// SURVEY.md §8(a)) and H^T (backprojection, steps B2-B3).  No tensor cores: the path is a gather /
// interpolate / accumulate over sphere-surface samples (Eq. 12, Eq. 36-39, Alg. 4) and its
// transpose (Eq. 23, Alg. 6), not a dense contraction.
//
// Work item = PATCH (transducer q, band of 32 time samples, block of 32 rings, azimuth sector of <= 32 directions): a
// compact piece of shell.  Patches are generated, culled and Morton-sorted once per geometry (oat_kernels.cu), so the
// blocks in flight work inside the same sub-volume and what they read / add into stays in L2.
//
// Register marching (round 2).  One block of 128 threads per patch, NO shared-memory ray list: warp w takes ring
// rows w, w+4, ..; lane = azimuth; every lane builds ITS ray in registers (direction from the fp64 table, fp64
// anchor at the band's mid radius, split into an integer node offset and a fraction in [-0.5, 0.5]) and marches it:
//   position   t_k = fma(u*step, k - 15.5, anchor_frac): ONE fp32 rounding at |t| < ~6 voxels (3e-7 voxel); this is
//              what keeps H within 1e-5 of the fp64 oracle after the time difference amplifies errors ~30x
//   cell       floor by a round-down add of 1.5*2^23; the cell's linear index is two integer multiply-adds away from
//              the three floats' bit patterns (all biases folded into one per-ray constant)
// The block holds ~1 KB of shared memory, so nearly all of the SM's 228 KB is L1 for the scattered record loads
// (measured: a 10-lane scattered request costs 12 SM-cycles below 8 KB of shared memory per block, 31 above 12 KB).
// H and H^T compute positions, cells and fractions with the same expressions, so they visit identical samples with
// identical weights (Eq. 12 vs Eq. 23).
#include "oat_internal.h"

#include <math.h>

namespace {

// floor() without the conversion pipe: adding 1.5*2^23 with round-toward-minus-infinity leaves floor(t) in the low
// mantissa bits (|t| < 2^22), so the integer is one integer add away from the float's bit pattern and floor(t) as a
// float is one exact subtraction away.
#define OAT_MAGIC 12582912.0f
#define OAT_MAGIC_BITS 0x4B400000u

struct RingRow {       // one ring of the patch, prepared once per patch by warp 0
    long long dofs;    // index of the sector's first direction in the direction table
    double ct;         // cos(theta_i)
    float omega;       // solid-angle weight (S2)
    int nj;            // directions of this ring in the patch's azimuth sector (0: ring not in the patch)
};

struct Ray {
    float ax, ay, az;  // anchor fraction in [-0.5, 0.5]
    float sx, sy, sz;  // direction * (voxels per time sample)
    float om;          // omega
    int ix, iy, iz;    // anchor node (padded node coordinates)
};

__device__ __forceinline__ void unpack_item(unsigned long long v, int &q, int &b, int &rb, int &s)
{
    s = (int)(v & 0xffffu);
    rb = (int)((v >> 16) & 0x3ffu);
    b = (int)((v >> 26) & 0xfffu);
    q = (int)(v >> 38);
}

// Direction (S3) of table entry d = sin(theta_i) (cos phi_j, sin phi_j) in the frame of the transducer, and the
// ray's anchor point base' + s_mid*u, all in fp64; returns false when the bounding box of the ray segment
// [s_lo, s_hi] cannot meet the padded node box.
__device__ __forceinline__ bool make_ray(const OatDev &P, double2 d, double ct, float omega, float stepf,
                                         const double *s_frame, Ray &e)
{
    float uu[3], af[3];
    int ai[3];
    bool hit = true;
    const float lim[3] = {(float)P.nx + 1.01f, (float)P.ny + 1.01f, (float)P.nz + 1.01f};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double ua = d.x * s_frame[a] + d.y * s_frame[3 + a] + ct * s_frame[6 + a];
        const double an = s_frame[9 + a] + s_frame[12] * ua;      // s_frame[12..14] = the band's s_mid, s_lo, s_hi
        const double ar = rint(an);
        uu[a] = (float)ua;
        af[a] = (float)(an - ar);
        ai[a] = (int)ar;
        const float p0 = (float)(s_frame[9 + a] + s_frame[13] * ua);
        const float p1 = (float)(s_frame[9 + a] + s_frame[14] * ua);
        hit = hit && (fmaxf(p0, p1) >= -0.01f) && (fminf(p0, p1) <= lim[a]);
    }
    e.ax = af[0]; e.ay = af[1]; e.az = af[2];
    e.sx = uu[0] * stepf; e.sy = uu[1] * stepf; e.sz = uu[2] * stepf;
    e.om = omega;
    e.ix = ai[0]; e.iy = ai[1]; e.iz = ai[2];
    return hit;
}

// warp 0 prepares the patch's 32 ring rows: the azimuth range [j0, j1) of sector `sec` of S in every ring
__device__ __forceinline__ void fill_ring_rows(const OatRing *__restrict__ ring, long long dir_ofs, int r0, int r1, int sec, int S,
                                               int lane, RingRow *s_ring)
{
    const int r = r0 + lane;
    RingRow row;
    row.dofs = 0; row.ct = 1.0; row.omega = 0.f; row.nj = 0;
    if (r < r1) {
        const OatRing R = ring[r];
        const int j0 = (int)(((long long)R.N * sec + S - 1) / S);
        const int j1 = (int)(((long long)R.N * (sec + 1) + S - 1) / S);
        row.dofs = dir_ofs + R.cum + j0;
        row.ct = R.ct;
        row.omega = R.omega;
        row.nj = j1 - j0;
    }
    s_ring[lane] = row;
}

__device__ __forceinline__ void prefetch_l1(const void *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

#define OAT_LDHINT ".L1::no_allocate"
__device__ __forceinline__ void ldg256_if(float (&c)[8], const float4 *p, bool pred)
{
    asm("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %9, 0;\n\t"
        "@p ld.global.nc" OAT_LDHINT ".v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t}"   // a record is used by one ray only
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]), "+f"(c[4]), "+f"(c[5]), "+f"(c[6]), "+f"(c[7])
        : "l"(p), "r"((int)pred));
}

// The two reductions of one marching step of H^T: quad L into record `cur` when `fl`, quad H into record `cur + sa` when `fh`
// (records of 16 bytes from `base`).  One 32 x 32 -> 64 bit multiply-add per address instead of 64-bit index arithmetic.
__device__ __forceinline__ void red_quads(unsigned long long base, unsigned cur, unsigned sa, bool fl, bool fh,
                                          float L0, float L1, float L2, float L3, float H0, float H1, float H2, float H3)
{
    asm volatile("{\n\t.reg .pred p, q;\n\t.reg .b64 a, b;\n\t.reg .b32 c2;\n\t"
                 "setp.ne.b32 p, %3, 0;\n\tsetp.ne.b32 q, %4, 0;\n\t"
                 "mad.wide.u32 a, %1, 16, %0;\n\t"
                 "add.u32 c2, %1, %2;\n\t"
                 "mad.wide.u32 b, c2, 16, %0;\n\t"
                 "@p red.global.add.v4.f32 [a], {%5,%6,%7,%8};\n\t"
                 "@q red.global.add.v4.f32 [b], {%9,%10,%11,%12};\n\t}"
                 ::"l"(base), "r"(cur), "r"(sa), "r"((int)fl), "r"((int)fh),
                   "f"(L0), "f"(L1), "f"(L2), "f"(L3), "f"(H0), "f"(H1), "f"(H2), "f"(H3) : "memory");
}

// sum acc[i] over the 16 lanes of each half-warp; lane l returns the total of acc[l & 15] of its half (15 shuffles)
__device__ __forceinline__ float half_warp_transpose_sum(float (&acc)[16], int lane)
{
#pragma unroll
    for (int s = 8; s >= 1; s >>= 1) {
        const bool up = (lane & s) != 0;
#pragma unroll
        for (int i = 0; i < s; ++i) {
            const float send = up ? acc[i] : acc[i + s];
            const float keep = up ? acc[i + s] : acc[i];
            acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, s);
        }
    }
    return acc[0];
}

// ------------------------------------------------------------------------------------------------
// Per-warp ray queue.  Only ~45 % of a patch's 1024 candidate directions survive the box cull (patches on the faces of
// the volume), so rays are compacted before they are marched: the lanes that built a surviving ray append it to a small
// ring buffer in shared memory owned by their warp (ballot + popc give the slot; no atomics, no block barrier), and the
// warp marches full groups from the front.  The buffers are the only sizeable shared memory of a block (6 KB for H), so
// the L1 carve-out stays at 64 KB per SM.
// ------------------------------------------------------------------------------------------------
// queue entry = two float4 kept in separate arrays (16-byte stride: conflict-free LDS.128 / STS.128):
//   a = anchor fraction (x, y, z), omega;  s = direction * step (x, y, z), then H: record-index constant K,
//   H^T: packed anchor node offsets

#define OAT_PB 128   // bias of the 10-bit packed anchor node offsets (H^T): offsets in [-128, 895], checked at create

// ------------------------------------------------------------------------------------------------
// H (projection).  A group of 16 queued rays is marched by all 32 lanes: lanes 0..15 take samples 0..15 of ray l,
// lanes 16..31 samples 31..16 of the same ray walked BACKWARDS with the direction negated -- fma(-s, -kk, a) ==
// fma(s, kk, a), so both halves run the same instruction stream with the same immediates kk = k' - 15.5 and the
// positions are bit-identical to a forward walk.  16 accumulators per lane (sample k' of the lower half, 31 - k' of the
// upper) fit the 56-register budget of 9 resident blocks per SM.
// Per step: 3 FFMA (position), 3 FADD.RM (floor), 1 IADD + 2 IMAD (record index), 1 ISETP (new cell?), 1 IMAD.WIDE,
// 1 predicated 256-bit load of the cell's polynomial record -- only when the ray has entered a new cell, ~2.2 samples
// share one load --, 6 FADD (fractions), 7 FFMA (Horner in fx, fy, fz) + 1 FFMA (quadrature weight): 26 instructions.
// The records carry a zero margin of P.cm cells around the padded box, so no sample needs a bounds test.
// ------------------------------------------------------------------------------------------------
#define OAT_NRH 1     // rays marched together by one lane (2 was measured: 92 registers, 24 warps per SM, slower)
#define OAT_QNH (16 * OAT_NRH + 32)    // queue entries per warp: at most 16 NRH - 1 left over + 32 new
#define OAT_MBLKH (1152 / OAT_MT)   // 9 blocks = 36 warps at 56 registers, no spills (8 blocks: 57.5 ms, 9: 54.6, 10: spills, 57.3)
__global__ void __launch_bounds__(OAT_MT, OAT_MBLKH)
oat_march_fwd_kernel(const OatDev P, const float4 *__restrict__ cells, float *__restrict__ y_out, double *__restrict__ g)
{
    __shared__ double s_frame[16];
    __shared__ RingRow s_ring[OAT_RI];
    __shared__ float4 s_qa[OAT_MT / 32][OAT_QNH], s_qs[OAT_MT / 32][OAT_QNH];
    __shared__ int s_flag;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float stepf = (float)P.step;
    const unsigned cx = (unsigned)P.cx, cxy = (unsigned)P.cxy;
    const unsigned kbias = (unsigned)P.cm - OAT_MAGIC_BITS;            // per axis: + margin - bias of the magic add
    const unsigned k_zero = 0u - OAT_MAGIC_BITS * (cxy + cx + 1u);     // ray (a = 0, s = 0) -> record 0 (all zero)
    const unsigned lt_mask = (1u << lane) - 1u;
    float4 *const qa = s_qa[warp], *const qs = s_qs[warp];
    for (long long item = blockIdx.x; item < P.n_patches; item += gridDim.x) {
        int q, b, rb, sec;
        unpack_item(P.patches[item], q, b, rb, sec);
        if (tid < 12) s_frame[tid] = P.frame[(size_t)q * 12 + tid];
        const OatBand band = P.band[b];
        if (tid == 32) { s_frame[12] = band.s_mid; s_frame[13] = (double)band.s_lo; s_frame[14] = (double)band.s_hi; }
        const double2 *__restrict__ dir = P.dir;
        const int r0 = rb * OAT_RI;
        const int r1 = min(r0 + OAT_RI, P.qb_rings[(size_t)q * P.NB + b]);
        if (warp == 0) fill_ring_rows(P.ring + band.ring_ofs, band.dir_ofs, r0, r1, sec, P.rb_sectors[band.rb_ofs + rb], lane, s_ring);
        float acc[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = 0.f;
        __syncthreads();
        // the directions of the NEXT ring row are prefetched into L1 while the current one is built and marched
        { const RingRow rw = s_ring[warp]; if (lane < rw.nj) prefetch_l1(dir + rw.dofs + lane); }
        int head = 0, cnt = 0;                                 // warp-uniform: first queued entry, number queued
#pragma unroll 1
        for (int rr = warp;; rr += OAT_MT / 32) {
            const bool last = rr >= OAT_RI;
            if (!last) {
                // ------------------------------------------------------------ build (A2: direction -> ray anchor)
                const RingRow row = s_ring[rr];
                if (rr + OAT_MT / 32 < OAT_RI) { const RingRow rw = s_ring[rr + OAT_MT / 32]; if (lane < rw.nj) prefetch_l1(dir + rw.dofs + lane); }
                if (row.nj > 0) {                               // warp-uniform
                    Ray e;
                    bool ok = lane < row.nj;
                    const double2 d = dir[row.dofs + (ok ? lane : 0)];
                    ok = make_ray(P, d, row.ct, row.omega, stepf, s_frame, e) && ok;
                    const unsigned m = __ballot_sync(0xffffffffu, ok);
                    if (ok) {
                        int slot = head + cnt + __popc(m & lt_mask);
                        if (slot >= OAT_QNH) slot -= OAT_QNH;
                        const unsigned K = ((unsigned)e.iz + kbias) * cxy + ((unsigned)e.iy + kbias) * cx + ((unsigned)e.ix + kbias);
                        qa[slot] = make_float4(e.ax, e.ay, e.az, e.om);
                        qs[slot] = make_float4(e.sx, e.sy, e.sz, __uint_as_float(K));
                    }
                    cnt += __popc(m);
                    __syncwarp();
                }
            }
            // ---------------------------------------------------------------- march (A3): groups of 16 * OAT_NRH rays
#pragma unroll 1
            while (cnt >= 16 * OAT_NRH || (last && cnt > 0)) {
                const int n = min(cnt, 16 * OAT_NRH);
                float ax[OAT_NRH], ay[OAT_NRH], az[OAT_NRH], om[OAT_NRH], sx[OAT_NRH], sy[OAT_NRH], sz[OAT_NRH];
                unsigned Kr[OAT_NRH], prev[OAT_NRH];
                float c[OAT_NRH][8];
#pragma unroll
                for (int r = 0; r < OAT_NRH; ++r) {
                    const int li = (lane & 15) + 16 * r;
                    int slot = head + li;
                    if (slot >= OAT_QNH) slot -= OAT_QNH;
                    float4 ea = make_float4(0.f, 0.f, 0.f, 0.f), es = make_float4(0.f, 0.f, 0.f, __uint_as_float(k_zero));
                    if (li < n) { ea = qa[slot]; es = qs[slot]; }
                    ax[r] = ea.x; ay[r] = ea.y; az[r] = ea.z; om[r] = ea.w;
                    sx[r] = lane >= 16 ? -es.x : es.x; sy[r] = lane >= 16 ? -es.y : es.y; sz[r] = lane >= 16 ? -es.z : es.z;
                    Kr[r] = __float_as_uint(es.w);
                    prev[r] = 0xffffffffu;                      // never a record index (those are < 2^31)
#pragma unroll
                    for (int i = 0; i < 8; ++i) c[r][i] = 0.f;
                }
                __syncwarp();                                   // the slots may be refilled by the next build
                head += n; if (head >= OAT_QNH) head -= OAT_QNH;
                cnt -= n;
#pragma unroll
                for (int k = 15; k >= 0; --k) {            // from the middle of the ray outwards: both halves start in (nearly) the same cell, one sector request
                    const float kk = (float)k - 15.5f;
                    float tx[OAT_NRH], ty[OAT_NRH], tz[OAT_NRH], rx[OAT_NRH], ry[OAT_NRH], rz[OAT_NRH];
#pragma unroll
                    for (int r = 0; r < OAT_NRH; ++r) {         // the loads of the lane's rays are in flight together
                        tx[r] = fmaf(sx[r], kk, ax[r]); ty[r] = fmaf(sy[r], kk, ay[r]); tz[r] = fmaf(sz[r], kk, az[r]);
                        rx[r] = __fadd_rd(tx[r], OAT_MAGIC); ry[r] = __fadd_rd(ty[r], OAT_MAGIC); rz[r] = __fadd_rd(tz[r], OAT_MAGIC);
                        const unsigned idx = __float_as_uint(rz[r]) * cxy + (__float_as_uint(ry[r]) * cx + (__float_as_uint(rx[r]) + Kr[r]));
                        const bool ch = idx != prev[r];
                        prev[r] = idx;
                        ldg256_if(c[r], cells + 2 * (size_t)idx, ch);
                    }
#pragma unroll
                    for (int r = 0; r < OAT_NRH; ++r) {
                        const float fx = tx[r] - (rx[r] - OAT_MAGIC), fy = ty[r] - (ry[r] - OAT_MAGIC), fz = tz[r] - (rz[r] - OAT_MAGIC);
                        // record = (c0, c4, c1, c5, c2, c6, c3, c7) of A = c0 + c1 fx + c2 fy + c3 fx fy + fz (c4 + c5 fx + c6 fy + c7 fx fy)
                        const float lo = fmaf(fy, fmaf(fx, c[r][6], c[r][4]), fmaf(fx, c[r][2], c[r][0]));
                        const float hi = fmaf(fy, fmaf(fx, c[r][7], c[r][5]), fmaf(fx, c[r][3], c[r][1]));
                        acc[k] = fmaf(om[r], fmaf(fz, hi, lo), acc[k]);
                    }
                }
            }
            if (last) break;
        }
        // S5: half-warp sums -> fp64 cross-warp combine -> one fp64 atomic per time sample
        const float tot = half_warp_transpose_sum(acc, lane);
        // the warps' partial sums go through the (now empty) ray queues
        float *const s_red = reinterpret_cast<float *>(s_qa);       // [warp][32] at a stride of OAT_QNH float4
        s_red[warp * (OAT_QNH * 4) + (lane < 16 ? lane : 47 - lane)] = tot;   // lane l >= 16 holds sample 31 - (l - 16)
        __syncthreads();
        if (warp == 0) {
            double sum = 0.0;
#pragma unroll
            for (int w = 0; w < OAT_MT / 32; ++w) sum += (double)s_red[w * (OAT_QNH * 4) + lane];
            const int k = band.k0 + lane;
            const double rho = P.c * (P.t0 + (double)k * P.dt);
            if (lane < band.nk && rho > 0.0 && sum != 0.0) atomicAdd(&g[(size_t)q * P.K + k], rho * rho * sum);
            // Fused step A4 (Eq. 3 L63 / Eq. 13): the block that completes the LAST patch of transducer q turns
            // the finished fp64 row g[q,:] into pressure.  Every lane fences its own atomics, one lane counts.
            __threadfence();
            __syncwarp();
            if (lane == 0) s_flag = (atomicAdd(&P.q_done[q], 1) + 1 == P.q_count[q]) ? 1 : 0;
        }
        __syncthreads();
        if (s_flag) {
            __threadfence();
            const double *gq = g + (size_t)q * P.K;
            float *yq = y_out + (size_t)q * P.K;
            for (int k = tid; k < P.K; k += OAT_MT) {
                double sp = 0.0, sm = 0.0;
                if (k + 1 < P.K) { const double t = P.t0 + (double)(k + 1) * P.dt; if (t > 0.0) sp = __ldcg(gq + k + 1) / t; }
                if (k - 1 >= 0) { const double t = P.t0 + (double)(k - 1) * P.dt; if (t > 0.0) sm = __ldcg(gq + k - 1) / t; }
                yq[k] = (float)(P.kappa * (sp - sm) / (2.0 * P.dt));
            }
        }
        __syncthreads();                                   // s_frame, s_ring, s_red, s_flag are reused by the next item
    }
}

// ------------------------------------------------------------------------------------------------
// H^T (backprojection), face-carrying form.  H^T is bound by the rate at which vector reductions retire in L2
// (~1.5 SM-cycles per RED.128 lane on scattered sectors, measured), so the aim is FEWER reductions per sample:
//   * one lane per queued ray, local axis 0 = the ray's dominant axis a (|u_a| largest), marched in the direction in
//     which the ray ADVANCES along a (backwards in k when u_a < 0; positions are identical, see above);
//   * the 8 corner weights of the current cell are accumulated as two quads, L on plane i_a and H on plane i_a + 1,
//     laid out as the face-quad records of orientation a (OatDev::f_base);
//   * when the ray steps to the next cell along a only (record index + one plane), the finished quad L is retired with
//     ONE reduction and H is carried over as the new L; any other cell change flushes both quads.
// ------------------------------------------------------------------------------------------------
#define OAT_MBLKT 9     // 55 registers, no spills; with 4 steps per loop trip: 77.7 -> 77.0 ms on the 512-transducer subset
#define OAT_QNT 64    // queue entries per warp: at most 31 left over + 32 new
__global__ void __launch_bounds__(OAT_MT, OAT_MBLKT)
oat_march_bwd_kernel(const OatDev P, float4 *__restrict__ faces, const float *__restrict__ y)
{
    __shared__ double s_frame[16];
    __shared__ RingRow s_ring[OAT_RI];
    __shared__ float4 s_qa[OAT_MT / 32][OAT_QNT], s_qs[OAT_MT / 32][OAT_QNT];
    __shared__ float s_coef[64];
    __shared__ int s_flag;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float stepf = (float)P.step;
    const unsigned lt_mask = (1u << lane) - 1u;
    float4 *const qa = s_qa[warp], *const qs = s_qs[warp];
    for (long long item = blockIdx.x; item < P.n_patches; item += gridDim.x) {
        int q, b, rb, sec;
        unpack_item(P.patches[item], q, b, rb, sec);
        if (tid < 12) s_frame[tid] = P.frame[(size_t)q * 12 + tid];
        const OatBand band = P.band[b];
        if (tid == 32) { s_frame[12] = band.s_mid; s_frame[13] = (double)band.s_lo; s_frame[14] = (double)band.s_hi; }
        const double2 *__restrict__ dir = P.dir;
        const int r0 = rb * OAT_RI;
        const int r1 = min(r0 + OAT_RI, P.qb_rings[(size_t)q * P.NB + b]);
        if (warp == 0) fill_ring_rows(P.ring + band.ring_ofs, band.dir_ofs, r0, r1, sec, P.rb_sectors[band.rb_ofs + rb], lane, s_ring);
        if (warp == 1) {
            // B1 fused at load (Eq. 22, S7 with the rho^2 of S8): the band's 32 coefficients
            // g'_k rho_k^2 = kappa (y[k-1] - y[k+1]) / (2 dt) / t_k * rho_k^2 straight from the data row (zero extension at both
            // ends, 0 where t_k <= 0), in fp64 with one rounding; stored forward and reversed
            float cf = 0.f;
            if (lane < band.nk) {
                const int k = band.k0 + lane;
                const float *__restrict__ row = y + (size_t)q * P.K;
                const double tk = P.t0 + (double)k * P.dt, rho = P.c * tk;
                const float ym = (k - 1 >= 0) ? row[k - 1] : 0.f;
                const float yp = (k + 1 < P.K) ? row[k + 1] : 0.f;
                const double sp = P.kappa * ((double)ym - (double)yp) / (2.0 * P.dt);
                cf = rho > 0.0 ? (float)(sp / tk * rho * rho) : 0.f;
            }
            s_coef[lane] = cf;
            s_coef[63 - lane] = cf;
            const bool any = __any_sync(0xffffffffu, cf != 0.f);
            if (lane == 0) s_flag = any ? 1 : 0;
        }
        __syncthreads();
        // a band whose 32 data values give g' = 0 contributes exactly nothing to H^T y
        if (s_flag != 0) {
            { const RingRow rw = s_ring[warp]; if (lane < rw.nj) prefetch_l1(dir + rw.dofs + lane); }
            int head = 0, cnt = 0;
#pragma unroll 1
            for (int rr = warp;; rr += OAT_MT / 32) {
                const bool last = rr >= OAT_RI;
                if (!last) {
                    const RingRow row = s_ring[rr];
                    if (rr + OAT_MT / 32 < OAT_RI) { const RingRow rw = s_ring[rr + OAT_MT / 32]; if (lane < rw.nj) prefetch_l1(dir + rw.dofs + lane); }
                    if (row.nj > 0) {                           // warp-uniform
                        Ray e;
                        bool ok = lane < row.nj;
                        const double2 d = dir[row.dofs + (ok ? lane : 0)];
                        ok = make_ray(P, d, row.ct, row.omega, stepf, s_frame, e) && ok;
                        const unsigned m = __ballot_sync(0xffffffffu, ok);
                        if (ok) {
                            const int slot = (head + cnt + __popc(m & lt_mask)) & (OAT_QNT - 1);
                            const unsigned pk = (unsigned)(e.ix + OAT_PB) | ((unsigned)(e.iy + OAT_PB) << 10) | ((unsigned)(e.iz + OAT_PB) << 20);
                            qa[slot] = make_float4(e.ax, e.ay, e.az, e.om);
                            qs[slot] = make_float4(e.sx, e.sy, e.sz, __uint_as_float(pk));
                        }
                        cnt += __popc(m);
                        __syncwarp();
                    }
                }
#pragma unroll 1
                while (cnt >= 32 || (last && cnt > 0)) {
                    const int n = min(cnt, 32);
                    const int slot = (head + lane) & (OAT_QNT - 1);
                    float4 ea = make_float4(0.f, 0.f, 0.f, 0.f), es = make_float4(1.f, 0.f, 0.f, 0.f);
                    if (lane < n) { ea = qa[slot]; es = qs[slot]; }
                    __syncwarp();
                    head = (head + n) & (OAT_QNT - 1);
                    cnt -= n;
                    const unsigned pk = __float_as_uint(es.w);
                    // anchor node offsets with the bias of the magic add folded in; an idle lane (lane >= n) gets -10^6: never valid
                    const int ex = lane < n ? (int)(pk & 1023u) - (int)(OAT_PB + OAT_MAGIC_BITS) : -1000000 - (int)OAT_MAGIC_BITS;
                    const int ey = (int)((pk >> 10) & 1023u) - (int)(OAT_PB + OAT_MAGIC_BITS), ez = (int)((pk >> 20) & 1023u) - (int)(OAT_PB + OAT_MAGIC_BITS);
                    const float mx = fabsf(es.x), my = fabsf(es.y), mz = fabsf(es.z);
                    const int o = (mx >= my && mx >= mz) ? 0 : (my >= mz ? 1 : 2);
                    // local axes (0, 1, 2) = (a, b, c) = (x,y,z), (y,z,x), (z,x,y)
                    const float a0 = o == 0 ? ea.x : o == 1 ? ea.y : ea.z, a1 = o == 0 ? ea.y : o == 1 ? ea.z : ea.x,
                                a2 = o == 0 ? ea.z : o == 1 ? ea.x : ea.y;
                    const float u0 = o == 0 ? es.x : o == 1 ? es.y : es.z, u1 = o == 0 ? es.y : o == 1 ? es.z : es.x,
                                u2 = o == 0 ? es.z : o == 1 ? es.x : es.y;
                    const int b0 = o == 0 ? ex : o == 1 ? ey : ez, b1 = o == 0 ? ey : o == 1 ? ez : ex, b2 = o == 0 ? ez : o == 1 ? ex : ey;
                    const unsigned n0 = o == 0 ? P.nx : o == 1 ? P.ny : P.nz, n1 = o == 0 ? P.ny : o == 1 ? P.nz : P.nx,
                                   n2 = o == 0 ? P.nz : o == 1 ? P.nx : P.ny;
                    const int nb = o == 0 ? P.f_nb[0] : o == 1 ? P.f_nb[1] : P.f_nb[2];
                    const int nc = o == 0 ? P.f_nc[0] : o == 1 ? P.f_nc[1] : P.f_nc[2];
                    const unsigned long long qb = (unsigned long long)(faces + (o == 0 ? P.f_base[0] : o == 1 ? P.f_base[1] : P.f_base[2]));
                    const int sa = nb * nc;                            // records per plane
                    const bool flip = u0 < 0.f;
                    const float s0 = flip ? -u0 : u0, s1 = flip ? -u1 : u1, s2 = flip ? -u2 : u2;   // s0 >= 0: the ray advances along local axis 0
                    const float *cp = s_coef + (flip ? 32 : 0);        // [0,32): coef_k, [32,64): coef_{31-k}
                    const float om = ea.w;
                    float L0 = 0.f, L1 = 0.f, L2 = 0.f, L3 = 0.f, H0 = 0.f, H1 = 0.f, H2 = 0.f, H3 = 0.f;
                    unsigned cur = 0;                                  // record index within orientation o (32-bit: one IMAD.WIDE per reduction)
                    bool valid = false;
                    // OAT_BU (4) steps per trip of a rolled loop: the fully unrolled body misses the instruction cache
#pragma unroll 1
                    for (int kb = 0; kb < 32; kb += OAT_BU) {
                        const float kbase = (float)kb - 15.5f;
#pragma unroll
                        for (int kj = 0; kj < OAT_BU; ++kj) {
                            const int k = kb + kj;
                            const float kk = kbase + (float)kj;
                            const float t0 = fmaf(s0, kk, a0), t1 = fmaf(s1, kk, a1), t2 = fmaf(s2, kk, a2);
                            const float r0f = __fadd_rd(t0, OAT_MAGIC), r1f = __fadd_rd(t1, OAT_MAGIC), r2f = __fadd_rd(t2, OAT_MAGIC);
                            const int i0 = __float_as_int(r0f) + b0, i1 = __float_as_int(r1f) + b1, i2 = __float_as_int(r2f) + b2;
                            const unsigned nxt = (unsigned)((i0 * nc + i2) * nb + i1);
                            const unsigned dcur = nxt - cur;
                            const bool chg = dcur != 0u;
                            const bool carry = dcur == (unsigned)sa;       // one cell forward along the dominant axis only
                            red_quads(qb, cur, (unsigned)sa, valid & chg, valid & chg & !carry, L0, L1, L2, L3, H0, H1, H2, H3);
                            L0 = chg ? (carry ? H0 : 0.f) : L0; L1 = chg ? (carry ? H1 : 0.f) : L1;
                            L2 = chg ? (carry ? H2 : 0.f) : L2; L3 = chg ? (carry ? H3 : 0.f) : L3;
                            H0 = chg ? 0.f : H0; H1 = chg ? 0.f : H1; H2 = chg ? 0.f : H2; H3 = chg ? 0.f : H3;
                            cur = nxt;
                            // padded cell n' in [0, N] <=> xi in [-1, N): the sample touches at least one existing node (S4)
                            valid = ((unsigned)i0 <= n0) & ((unsigned)i1 <= n1) & ((unsigned)i2 <= n2);
                            const float f0 = t0 - (r0f - OAT_MAGIC), f1 = t1 - (r1f - OAT_MAGIC), f2 = t2 - (r2f - OAT_MAGIC);
                            const float cw = valid ? cp[k] * om : 0.f;
                            const float e1 = 1.f - f1, e2 = 1.f - f2;
                            const float q0 = e1 * e2, q1 = f1 * e2, q2 = e1 * f2, q3 = f1 * f2;
                            const float wh = cw * f0, wl = cw - wh;
                            L0 = fmaf(q0, wl, L0); L1 = fmaf(q1, wl, L1); L2 = fmaf(q2, wl, L2); L3 = fmaf(q3, wl, L3);
                            H0 = fmaf(q0, wh, H0); H1 = fmaf(q1, wh, H1); H2 = fmaf(q2, wh, H2); H3 = fmaf(q3, wh, H3);
                        }
                    }
                    red_quads(qb, cur, (unsigned)sa, valid, valid, L0, L1, L2, L3, H0, H1, H2, H3);
                }
                if (last) break;
            }
        }
        __syncthreads();                                   // s_frame, s_ring, s_coef, s_flag are reused by the next item
    }
}

// cell records from x: record of cell (X,Y,Z) of the margin-extended array, X in [0, cx) etc.; padded cell index
// ix = X - cm in [0, nx] has the corner nodes ix-1..ix in real indices (zero outside the grid = reading G5; the margin
// records are all zero).  A record holds the coefficients of the cell's trilinear polynomial
//   A(fx,fy,fz) = c0 + c1 fx + c2 fy + c3 fx fy + fz (c4 + c5 fx + c6 fy + c7 fx fy)        (Eq. 10 L110 expanded)
// computed in fp64 from the 8 corner values and rounded once to fp32, stored as (c0, c4, c1, c5, c2, c6, c3, c7).
__global__ void oat_pad_cells_kernel(const OatDev P, const float *__restrict__ x, float4 *__restrict__ cells)
{
    const long long n = (long long)P.cz * P.cxy;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double v[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        const int X = (int)(i % P.cx) - P.cm;
        const long long r = i / P.cx;
        const int Y = (int)(r % P.cy) - P.cm, Z = (int)(r / P.cy) - P.cm;
        bool any = false;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int xx = X - 1 + (k & 1), yy = Y - 1 + ((k >> 1) & 1), zz = Z - 1 + (k >> 2);
            if (xx >= 0 && xx < P.nx && yy >= 0 && yy < P.ny && zz >= 0 && zz < P.nz) {
                v[k] = (double)x[((size_t)zz * P.ny + yy) * P.nx + xx];
                any = true;
            }
        }
        if (!any) { cells[2 * i] = make_float4(0.f, 0.f, 0.f, 0.f); cells[2 * i + 1] = make_float4(0.f, 0.f, 0.f, 0.f); continue; }
        const double c1 = v[1] - v[0], c2 = v[2] - v[0], c4 = v[4] - v[0];
        const double c3 = v[3] - v[2] - c1, c5 = v[5] - v[4] - c1, c6 = v[6] - v[4] - c2;
        const double c7 = v[7] - v[6] - (v[5] - v[4]) - c3;
        cells[2 * i] = make_float4((float)v[0], (float)c4, (float)c1, (float)c5);
        cells[2 * i + 1] = make_float4((float)c2, (float)c6, (float)c3, (float)c7);
    }
}

}  // namespace

void oat_launch_pad_cells(const OatDev &P, const float *x, float4 *cells, cudaStream_t st)
{
    const long long n = (long long)P.cz * P.cxy;
    long long gsz = (n + 255) / 256;
    if (gsz > 148LL * 16) gsz = 148LL * 16;
    if (gsz < 1) gsz = 1;
    oat_pad_cells_kernel<<<(unsigned)gsz, 256, 0, st>>>(P, x, cells);
}

cudaError_t oat_launch_march(int mode, const OatDev &P, const float4 *cells, float4 *faces, float *y_out,
                             const float *y_in, double *g, cudaStream_t st)
{
    if (P.n_patches <= 0) return cudaSuccess;
    const long long cap = 0x7fffffffLL;
    const unsigned grid = (unsigned)(P.n_patches < cap ? P.n_patches : cap);
    if (mode == 0) oat_march_fwd_kernel<<<grid, OAT_MT, 0, st>>>(P, cells, y_out, g);
    else oat_march_bwd_kernel<<<grid, OAT_MT, 0, st>>>(P, faces, y_in);
    return cudaGetLastError();
}
