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
__device__ __forceinline__ bool make_ray(const OatDev &P, const OatBand &band, double2 d, double ct, float omega, float stepf,
                                         const double *s_frame, Ray &e)
{
    float uu[3], af[3];
    int ai[3];
    bool hit = true;
    const float lim[3] = {(float)P.nx + 1.01f, (float)P.ny + 1.01f, (float)P.nz + 1.01f};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double ua = d.x * s_frame[a] + d.y * s_frame[3 + a] + ct * s_frame[6 + a];
        const double an = s_frame[9 + a] + band.s_mid * ua;
        const double ar = rint(an);
        uu[a] = (float)ua;
        af[a] = (float)(an - ar);
        ai[a] = (int)ar;
        const float p0 = (float)(s_frame[9 + a] + (double)band.s_lo * ua);
        const float p1 = (float)(s_frame[9 + a] + (double)band.s_hi * ua);
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

__device__ __forceinline__ void ldg256_if(float (&c)[8], const float4 *p, bool pred)
{
    asm("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %9, 0;\n\t"
        "@p ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t}"   // a record is used by one ray only
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]), "+f"(c[4]), "+f"(c[5]), "+f"(c[6]), "+f"(c[7])
        : "l"(p), "r"((int)pred));
}

__device__ __forceinline__ void red_add_v4_if(float4 *addr, float a, float b, float c, float d, bool pred)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\t@p red.global.add.v4.f32 [%0], {%1,%2,%3,%4};\n\t}"
                 ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d), "r"((int)pred) : "memory");
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
// H (projection).  A ring row (<= 32 rays, lane = azimuth) is marched in two passes of 16 rays by all 32 lanes: lanes
// 0..15 take samples 0..15 of ray p*16 + l, lanes 16..31 samples 31..16 of the same ray walked BACKWARDS with the
// direction negated -- fma(-s, -kk, a) == fma(s, kk, a), so both halves run the same instruction stream with the same
// immediates kk = k' - 15.5 and the positions are bit-identical to a forward walk.  16 accumulators per lane
// (sample k' of the lower half, 31 - k' of the upper) fit the 64-register budget of 8 resident blocks per SM.
// Per step: 3 FFMA (position), 3 FADD.RM (floor), 1 IADD + 2 IMAD (record index), 1 ISETP (new cell?), 1 IMAD.WIDE,
// 1 predicated 256-bit load of the cell's polynomial record -- only when the ray has entered a new cell, ~2.2 samples
// share one load --, 6 FADD (fractions), 7 FFMA (Horner in fx, fy, fz) + 1 FFMA (quadrature weight): 26 instructions.
// The records carry a zero margin of P.cm cells around the padded box, so no sample needs a bounds test.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(OAT_MT, 8)
oat_march_fwd_kernel(const OatDev P, const float4 *__restrict__ cells, float *__restrict__ y_out, double *__restrict__ g)
{
    __shared__ double s_frame[12];
    __shared__ RingRow s_ring[OAT_RI];
    __shared__ float s_red[OAT_MT / 32][32];
    __shared__ int s_flag;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float stepf = (float)P.step;
    const unsigned cx = (unsigned)P.cx, cxy = (unsigned)P.cxy;
    const unsigned kbias = (unsigned)P.cm - OAT_MAGIC_BITS;            // per axis: + margin - bias of the magic add
    const unsigned k_zero = 0u - OAT_MAGIC_BITS * (cxy + cx + 1u);     // ray (a = 0, s = 0) -> record 0 (all zero)
    for (long long item = blockIdx.x; item < P.n_patches; item += gridDim.x) {
        int q, b, rb, sec;
        unpack_item(P.patches[item], q, b, rb, sec);
        if (tid < 12) s_frame[tid] = P.frame[(size_t)q * 12 + tid];
        const OatBand band = P.band[b];
        const double2 *__restrict__ dir = P.dir;
        const int r0 = rb * OAT_RI;
        const int r1 = min(r0 + OAT_RI, P.qb_rings[(size_t)q * P.NB + b]);
        if (warp == 0) fill_ring_rows(P.ring + band.ring_ofs, band.dir_ofs, r0, r1, sec, P.rb_sectors[band.rb_ofs + rb], lane, s_ring);
        float acc[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = 0.f;
        __syncthreads();
        // the direction of the NEXT ring row is loaded while the current one is marched
        double2 dn = make_double2(0.0, 0.0);
        if (warp < OAT_RI) { const RingRow rw = s_ring[warp]; if (lane < rw.nj) dn = dir[rw.dofs + lane]; }
#pragma unroll 1
        for (int rr = warp; rr < OAT_RI; rr += OAT_MT / 32) {
            const RingRow row = s_ring[rr];
            const double2 d = dn;
            if (rr + OAT_MT / 32 < OAT_RI) { const RingRow rw = s_ring[rr + OAT_MT / 32]; if (lane < rw.nj) dn = dir[rw.dofs + lane]; }
            if (row.nj <= 0) continue;                          // warp-uniform
            Ray e;
            bool ok = lane < row.nj;
            ok = make_ray(P, band, d, row.ct, row.omega, stepf, s_frame, e) && ok;
            unsigned K = ((unsigned)e.iz + kbias) * cxy + ((unsigned)e.iy + kbias) * cx + ((unsigned)e.ix + kbias);
            if (!ok) { e.ax = e.ay = e.az = 0.f; e.sx = e.sy = e.sz = 0.f; e.om = 0.f; K = k_zero; }
            const unsigned okm = __ballot_sync(0xffffffffu, ok);
#pragma unroll 1
            for (int pass = 0; pass < 2; ++pass) {
                if (((okm >> (16 * pass)) & 0xffffu) == 0u) continue;   // warp-uniform
                const int src = pass * 16 + (lane & 15);
                const float ax = __shfl_sync(0xffffffffu, e.ax, src), ay = __shfl_sync(0xffffffffu, e.ay, src),
                            az = __shfl_sync(0xffffffffu, e.az, src), om = __shfl_sync(0xffffffffu, e.om, src);
                float sx = __shfl_sync(0xffffffffu, e.sx, src), sy = __shfl_sync(0xffffffffu, e.sy, src),
                      sz = __shfl_sync(0xffffffffu, e.sz, src);
                const unsigned Kr = __shfl_sync(0xffffffffu, K, src);
                if (lane >= 16) { sx = -sx; sy = -sy; sz = -sz; }
                float c[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) c[i] = 0.f;
                unsigned prev = 0xffffffffu;                    // never a record index (those are < 2^31)
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    const float kk = (float)k - 15.5f;
                    const float tx = fmaf(sx, kk, ax), ty = fmaf(sy, kk, ay), tz = fmaf(sz, kk, az);
                    const float rx = __fadd_rd(tx, OAT_MAGIC), ry = __fadd_rd(ty, OAT_MAGIC), rz = __fadd_rd(tz, OAT_MAGIC);
                    const unsigned idx = __float_as_uint(rz) * cxy + (__float_as_uint(ry) * cx + (__float_as_uint(rx) + Kr));
                    const bool ch = idx != prev;
                    prev = idx;
                    ldg256_if(c, cells + 2 * (size_t)idx, ch);
                    const float fx = tx - (rx - OAT_MAGIC), fy = ty - (ry - OAT_MAGIC), fz = tz - (rz - OAT_MAGIC);
                    // record = (c0, c4, c1, c5, c2, c6, c3, c7) of A = c0 + c1 fx + c2 fy + c3 fx fy + fz (c4 + c5 fx + c6 fy + c7 fx fy)
                    const float lo = fmaf(fy, fmaf(fx, c[6], c[4]), fmaf(fx, c[2], c[0]));
                    const float hi = fmaf(fy, fmaf(fx, c[7], c[5]), fmaf(fx, c[3], c[1]));
                    acc[k] = fmaf(om, fmaf(fz, hi, lo), acc[k]);
                }
            }
        }
        // S5: half-warp sums -> fp64 cross-warp combine -> one fp64 atomic per time sample
        const float tot = half_warp_transpose_sum(acc, lane);
        s_red[warp][lane < 16 ? lane : 47 - lane] = tot;           // lane l >= 16 holds sample 31 - (l - 16)
        __syncthreads();
        if (warp == 0) {
            double sum = 0.0;
#pragma unroll
            for (int w = 0; w < OAT_MT / 32; ++w) sum += (double)s_red[w][lane];
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
//   * one lane per ray, local axis 0 = the ray's dominant axis a (|u_a| largest), marched in the direction in which
//     the ray ADVANCES along a (backwards in k when u_a < 0; positions are identical, see above);
//   * the 8 corner weights of the current cell are accumulated as two quads, L on plane i_a and H on plane i_a + 1,
//     laid out as the face-quad records of orientation a (OatDev::f_base);
//   * when the ray steps to the next cell along a only, the finished quad L is retired with ONE reduction and H is
//     carried over as the new L; only a step across one of the two minor axes flushes both quads.
// ------------------------------------------------------------------------------------------------
#ifndef OAT_MBLKT
#define OAT_MBLKT 6
#endif
__global__ void __launch_bounds__(OAT_MT, OAT_MBLKT)
oat_march_bwd_kernel(const OatDev P, float4 *__restrict__ faces, const float *__restrict__ coef)
{
    __shared__ double s_frame[12];
    __shared__ RingRow s_ring[OAT_RI];
    __shared__ float s_coef[64];
    __shared__ int s_flag;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float stepf = (float)P.step;
    for (long long item = blockIdx.x; item < P.n_patches; item += gridDim.x) {
        int q, b, rb, sec;
        unpack_item(P.patches[item], q, b, rb, sec);
        if (tid < 12) s_frame[tid] = P.frame[(size_t)q * 12 + tid];
        const OatBand band = P.band[b];
        const double2 *__restrict__ dir = P.dir;
        const int r0 = rb * OAT_RI;
        const int r1 = min(r0 + OAT_RI, P.qb_rings[(size_t)q * P.NB + b]);
        if (warp == 0) fill_ring_rows(P.ring + band.ring_ofs, band.dir_ofs, r0, r1, sec, P.rb_sectors[band.rb_ofs + rb], lane, s_ring);
        if (warp == 1) {                                   // B1: the band's 32 coefficients g'_k rho_k^2, forward and reversed
            const float cf = lane < band.nk ? coef[(size_t)q * P.K + band.k0 + lane] : 0.f;
            s_coef[lane] = cf;
            s_coef[63 - lane] = cf;
            const bool any = __any_sync(0xffffffffu, cf != 0.f);
            if (lane == 0) s_flag = any ? 1 : 0;
        }
        __syncthreads();
        // a band whose 32 data values give g' = 0 contributes exactly nothing to H^T y
        if (s_flag != 0) {
            double2 dn = make_double2(0.0, 0.0);
            if (warp < OAT_RI) { const RingRow rw = s_ring[warp]; if (lane < rw.nj) dn = dir[rw.dofs + lane]; }
#pragma unroll 1
            for (int rr = warp; rr < OAT_RI; rr += OAT_MT / 32) {
                const RingRow row = s_ring[rr];
                const double2 d = dn;
                if (rr + OAT_MT / 32 < OAT_RI) { const RingRow rw = s_ring[rr + OAT_MT / 32]; if (lane < rw.nj) dn = dir[rw.dofs + lane]; }
                if (row.nj <= 0) continue;                      // warp-uniform
                Ray e;
                bool ok = lane < row.nj;
                ok = make_ray(P, band, d, row.ct, row.omega, stepf, s_frame, e) && ok;
                if (!__any_sync(0xffffffffu, ok)) continue;
                if (!ok) { e.ax = e.ay = e.az = 0.f; e.sx = e.sy = e.sz = 0.f; e.ix = e.iy = e.iz = -1000; }   // never valid: no reduction
                const float mx = fabsf(e.sx), my = fabsf(e.sy), mz = fabsf(e.sz);
                const int o = (mx >= my && mx >= mz) ? 0 : (my >= mz ? 1 : 2);
                // local axes (0, 1, 2) = (a, b, c) = (x,y,z), (y,z,x), (z,x,y)
                const float a0 = o == 0 ? e.ax : o == 1 ? e.ay : e.az, a1 = o == 0 ? e.ay : o == 1 ? e.az : e.ax,
                            a2 = o == 0 ? e.az : o == 1 ? e.ax : e.ay;
                const float u0 = o == 0 ? e.sx : o == 1 ? e.sy : e.sz, u1 = o == 0 ? e.sy : o == 1 ? e.sz : e.sx,
                            u2 = o == 0 ? e.sz : o == 1 ? e.sx : e.sy;
                const int b0 = (o == 0 ? e.ix : o == 1 ? e.iy : e.iz) - (int)OAT_MAGIC_BITS, b1 = (o == 0 ? e.iy : o == 1 ? e.iz : e.ix) - (int)OAT_MAGIC_BITS,
                          b2 = (o == 0 ? e.iz : o == 1 ? e.ix : e.iy) - (int)OAT_MAGIC_BITS;
                const unsigned n0 = o == 0 ? P.nx : o == 1 ? P.ny : P.nz, n1 = o == 0 ? P.ny : o == 1 ? P.nz : P.nx,
                               n2 = o == 0 ? P.nz : o == 1 ? P.nx : P.ny;
                const int nb = o == 0 ? P.f_nb[0] : o == 1 ? P.f_nb[1] : P.f_nb[2];
                const int nc = o == 0 ? P.f_nc[0] : o == 1 ? P.f_nc[1] : P.f_nc[2];
                float4 *const qb = faces + (o == 0 ? P.f_base[0] : o == 1 ? P.f_base[1] : P.f_base[2]);
                const int sa = nb * nc;                            // records per plane
                const bool flip = u0 < 0.f;
                const float s0 = flip ? -u0 : u0, s1 = flip ? -u1 : u1, s2 = flip ? -u2 : u2;   // s0 >= 0: the ray advances along local axis 0
                const float *cp = s_coef + (flip ? 32 : 0);        // [0,32): coef_k, [32,64): coef_{31-k}
                const float om = ok ? e.om : 0.f;
                float L0 = 0.f, L1 = 0.f, L2 = 0.f, L3 = 0.f, H0 = 0.f, H1 = 0.f, H2 = 0.f, H3 = 0.f;
                float pr0 = 0.f, pr1 = 0.f, pr2 = 0.f;             // never equal to a rounded coordinate (those are >= 2^22)
                unsigned cur = 0;                                  // record index within orientation o
                bool valid = false;
                // 8 steps per trip of a rolled loop: the fully unrolled body missed the instruction cache
#pragma unroll 1
                for (int kb = 0; kb < 32; kb += OAT_BU) {
                    const float kbase = (float)kb - 15.5f;
#pragma unroll
                    for (int kj = 0; kj < OAT_BU; ++kj) {
                        const int k = kb + kj;
                        const float kk = kbase + (float)kj;
                        const float t0 = fmaf(s0, kk, a0), t1 = fmaf(s1, kk, a1), t2 = fmaf(s2, kk, a2);
                        const float r0f = __fadd_rd(t0, OAT_MAGIC), r1f = __fadd_rd(t1, OAT_MAGIC), r2f = __fadd_rd(t2, OAT_MAGIC);
                        const bool c12 = (r1f != pr1) | (r2f != pr2);
                        const bool c0 = r0f != pr0;
                        const bool carry = (!c12) & (r0f == pr0 + 1.0f);    // one cell forward along the dominant axis only
                        const bool full = c12 | (c0 & !carry);
                        red_add_v4_if(qb + cur, L0, L1, L2, L3, valid & (c0 | c12));
                        red_add_v4_if(qb + (cur + (unsigned)sa), H0, H1, H2, H3, valid & full);
                        L0 = full ? 0.f : (carry ? H0 : L0); L1 = full ? 0.f : (carry ? H1 : L1);
                        L2 = full ? 0.f : (carry ? H2 : L2); L3 = full ? 0.f : (carry ? H3 : L3);
                        const bool zh = full | carry;
                        H0 = zh ? 0.f : H0; H1 = zh ? 0.f : H1; H2 = zh ? 0.f : H2; H3 = zh ? 0.f : H3;
                        pr0 = r0f; pr1 = r1f; pr2 = r2f;
                        const int i0 = __float_as_int(r0f) + b0, i1 = __float_as_int(r1f) + b1, i2 = __float_as_int(r2f) + b2;
                        // padded cell n' in [0, N] <=> xi in [-1, N): the sample touches at least one existing node (S4)
                        valid = ((unsigned)i0 <= n0) & ((unsigned)i1 <= n1) & ((unsigned)i2 <= n2);
                        cur = (unsigned)((i0 * nc + i2) * nb + i1);
                        const float f0 = t0 - (r0f - OAT_MAGIC), f1 = t1 - (r1f - OAT_MAGIC), f2 = t2 - (r2f - OAT_MAGIC);
                        const float cwk = cp[k] * om;
                        const float cw = valid ? cwk : 0.f;
                        const float e1 = 1.f - f1, e2 = 1.f - f2;
                        const float q0 = e1 * e2, q1 = f1 * e2, q2 = e1 * f2, q3 = f1 * f2;
                        const float wh = cw * f0, wl = cw - wh;
                        L0 = fmaf(q0, wl, L0); L1 = fmaf(q1, wl, L1); L2 = fmaf(q2, wl, L2); L3 = fmaf(q3, wl, L3);
                        H0 = fmaf(q0, wh, H0); H1 = fmaf(q1, wh, H1); H2 = fmaf(q2, wh, H2); H3 = fmaf(q3, wh, H3);
                    }
                }
                red_add_v4_if(qb + cur, L0, L1, L2, L3, valid);
                red_add_v4_if(qb + (cur + (unsigned)sa), H0, H1, H2, H3, valid);
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
                             const float *coef, double *g, cudaStream_t st)
{
    if (P.n_patches <= 0) return cudaSuccess;
    const long long cap = 0x7fffffffLL;
    const unsigned grid = (unsigned)(P.n_patches < cap ? P.n_patches : cap);
    if (mode == 0) oat_march_fwd_kernel<<<grid, OAT_MT, 0, st>>>(P, cells, y_out, g);
    else oat_march_bwd_kernel<<<grid, OAT_MT, 0, st>>>(P, faces, coef);
    return cudaGetLastError();
}
