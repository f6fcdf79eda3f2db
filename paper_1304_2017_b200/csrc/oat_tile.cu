// Tile-stationary marching kernels of liboat.so for sm_100a (B200): SURVEY.md §8(a) candidate V2.
//
// The patch kernels of oat_march.cu read one 32-byte polynomial record per cell run from L2 (~14 B per sample, ~6 TB/s at
// config 3: the L2 -> SM path is what bounds them).  Here a block keeps a BRICK of the volume in shared memory and all
// samples that fall into it are evaluated from there, whatever transducer they belong to:
//
//   tile       a core of 16^3 cells (padded cell index) plus a margin of 3 cells on every side (22^3 cells)
//   records    per (cell column x, y; node plane z) the bilinear polynomial of the four nodes of that plane,
//              (v00, v10 - v00, v01 - v00, v11 - v10 - v01 + v00): 16 bytes, 23 planes x 22 x 22 = 182 KB of shared memory.
//              A sample in cell (x, y, z) is lo + fz (hi - lo) with lo / hi the polynomials of planes z / z + 1 (Eq. 10,
//              Eq. 12).  The raw nodes of the brick come in by TMA (3-D box of the caller's volume, out-of-bounds
//              elements filled with zero = the zero padding of reading G5), two half bricks staged through 26 KB
//   work unit  a CHUNK = 8 consecutive time samples of one ray (transducer q, band b, ring i, azimuth j).  A chunk belongs to
//              the tile whose CORE holds the cell of its first sample; 7 steps of <= 3/7 cell reach at most 3 cells further,
//              so every sample of an owned chunk finds its record in the brick and the marching loop needs no bounds test
//   schedule   persistent blocks (one per SM, 16 warps) take (tile, transducer range) items from a global counter; inside an
//              item every warp takes whole transducers: it finds the bands whose shells cross the core, the window of rings
//              and azimuths that covers the core's projection, builds the candidate rays (direction table -> fp32 cull
//              against the core -> fp64 anchor -> exact ownership test of the four chunks), compacts the owned chunks into
//              a per-warp queue and marches 32 of them at a time.  No block-wide barrier inside an item.
//
// Positions are those of oat_march.cu: t_k = fma(u * step, k - 15.5, anchor_frac) about the fp64 anchor at the band's mid
// radius, floor by the round-down add of 1.5 * 2^23; the ownership test uses the same expression, so every chunk has
// exactly one owner and H visits the sample set of OAT-DISC v1 exactly once.
#include "oat_internal.h"

#include <cuda.h>
#include <math.h>
#include <string.h>

namespace {

#define OAT_MAGIC 12582912.0f
#define OAT_MAGIC_BITS 0x4B400000u

#define TT_C 16                        // core cells per axis
#define TT_M 3                         // margin cells: floor(7 * step) + 1 <= 3  <=>  step < 3/7
#define TT_R (TT_C + 2 * TT_M)         // 22 cells per axis in the brick
#define TT_NP (TT_R + 1)               // 23 node planes
#define TT_PY (TT_R + 1)               // record pitch of a row (odd: neighbouring rows fall into different 16-byte bank groups)
#define TT_PZ (TT_PY * TT_R + 1)       // record pitch of a plane (odd mod 8)
#define TT_NREC (TT_NP * TT_PZ)        // float4 records
#define TT_WARPS 16
#define TT_THREADS (TT_WARPS * 32)
#define TT_QN 64                       // queue entries per warp: at most 31 left over + 32 new
#define TT_BX 24                       // staged box: 24 x 23 nodes per plane (x extent a multiple of 16 bytes),
#define TT_BY 23
#define TT_BZ 12                       // 12 planes per round
#define TT_STAGE_BYTES (TT_BX * TT_BY * TT_BZ * 4)
#define TT_QUEUE_BYTES (TT_WARPS * TT_QN * 32)
static_assert(TT_C % 4 == 0 && (2 * TT_M + 2) % 4 == 0 && TT_R + 2 <= TT_BX, "the staged box must start on a multiple of 4 nodes in x");

struct TileParams {
    int ntx, nty, ntz;                 // tiles per axis; tile t has the core cells [-TT_M + TT_C t, -TT_M + TT_C (t + 1))
    int n_qc, nq;                      // transducer ranges per tile, transducers per range
    long long n_items;
    int use_tma;
};

struct SmemLayout {
    float4 rec[TT_NREC];
    union alignas(128) {
        struct { float4 qa[TT_WARPS][TT_QN], qs[TT_WARPS][TT_QN]; } q;
        float stage[TT_BX * TT_BY * TT_BZ];
    } u;
    unsigned char qc[TT_WARPS][TT_QN];
    unsigned cq[TT_WARPS][TT_QN];      // candidate queue: ring slot << 27 | index into the band's direction table
    double frame[TT_WARPS][16];        // e_x, e_y, e_z, base', then the band's s_mid, s_lo, s_hi
    float framef[TT_WARPS][12];
    unsigned long long mbar;
    long long item;
    int nextq;
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 3-D box of the volume -> shared memory; elements outside the tensor arrive as zero (reading G5)
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, unsigned long long *bar, int x, int y, int z)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z) : "memory");
}

struct Ray {
    float ax, ay, az;  // anchor fraction in [-0.5, 0.5]
    float sx, sy, sz;  // direction * (voxels per time sample)
    int ix, iy, iz;    // anchor node (padded node coordinates)
};

// Direction (S3) of table entry d = sin(theta_i) (cos phi_j, sin phi_j) in the frame of the transducer and the ray's anchor
// base' + s_mid u in fp64 (the same arithmetic as oat_march.cu); false when the bounding box of the ray's segment
// [s_lo, s_hi] cannot meet the padded node box.
__device__ __forceinline__ bool make_ray(const OatDev &P, double2 d, double ct, float stepf, const double *s_frame, Ray &e)
{
    float uu[3], af[3];
    int ai[3];
    bool hit = true;
    const float lim[3] = {(float)P.nx + 1.01f, (float)P.ny + 1.01f, (float)P.nz + 1.01f};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double ua = d.x * s_frame[a] + d.y * s_frame[3 + a] + ct * s_frame[6 + a];
        const double an = s_frame[9 + a] + s_frame[12] * ua;
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
    e.ix = ai[0]; e.iy = ai[1]; e.iz = ai[2];
    return hit;
}

__device__ __forceinline__ void prefetch_l1(const void *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

__device__ __forceinline__ float warp_min(float v)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}
__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}

// sum v[i] over all 32 lanes for i = 0..7; lane l returns the total of v[l & 7] (7 + 2 shuffles)
__device__ __forceinline__ float warp_transpose_sum8(float (&v)[8], int lane)
{
#pragma unroll
    for (int s = 4; s >= 1; s >>= 1) {
        const bool up = (lane & s) != 0;
#pragma unroll
        for (int i = 0; i < s; ++i) {
            const float send = up ? v[i] : v[i + s];
            const float keep = up ? v[i + s] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, s);
        }
    }
    float r = v[0];
    r += __shfl_xor_sync(0xffffffffu, r, 8);
    r += __shfl_xor_sync(0xffffffffu, r, 16);
    return r;
}

// ------------------------------------------------------------------------------------------------
// March one group of <= 32 queued chunks (A3): lane = chunk, 8 samples each.  Per step: 3 FFMA (position), 3 FADD.RM
// (floor), 3 integer multiply-adds (shared-memory address of the cell's record), 2 predicated LDS.128 when the ray has
// entered a new cell, 6 FADD (fractions), 2 x 3 FFMA (bilinear polynomials of the two planes), 2 for the lerp in z, 1 for
// the quadrature weight.  The value of step i of a chunk with index c belongs to sample 8 c + i of the band: it is added to
// acc[c][i] through a 0/1 mask per chunk index (4 FFMA), so the accumulators are summed over lanes only once per band.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void lds_records_if_new(float4 &lo, float4 &hi, unsigned adr, unsigned &prev)
{
    asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %8, %9;\n\t"
        "@p ld.shared.v4.f32 {%0,%1,%2,%3}, [%8];\n\t"
        "@p ld.shared.v4.f32 {%4,%5,%6,%7}, [%8+%10];\n\t}"
        : "+f"(lo.x), "+f"(lo.y), "+f"(lo.z), "+f"(lo.w), "+f"(hi.x), "+f"(hi.y), "+f"(hi.z), "+f"(hi.w)
        : "r"(adr), "r"(prev), "n"(16 * TT_PZ));
    prev = adr;
}

__device__ __forceinline__ void march_group_fwd(const float4 *qa, const float4 *qs, const unsigned char *qc, int &head, int &cnt,
                                                float (&acc)[4][8], int lane, unsigned rec_base)
{
    const int n = min(cnt, 32);
    const int slot = (head + lane) & (TT_QN - 1);
    float4 ea = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 es = make_float4(0.f, 0.f, 0.f, __uint_as_float(rec_base - 16u * OAT_MAGIC_BITS * (1u + TT_PY + TT_PZ)));   // idle lane: cell 0, weight 0
    int cc = 0;
    if (lane < n) { ea = qa[slot]; es = qs[slot]; cc = qc[slot]; }
    __syncwarp();                                           // the slots may be refilled by the next build
    head = (head + n) & (TT_QN - 1);
    cnt -= n;
    const unsigned Kr = __float_as_uint(es.w);
    const float kk0 = 8.f * (float)cc - 15.5f;
    const float m0 = cc == 0 ? ea.w : 0.f, m1 = cc == 1 ? ea.w : 0.f, m2 = cc == 2 ? ea.w : 0.f, m3 = cc == 3 ? ea.w : 0.f;   // omega x [c == c']
    unsigned prev = 0xffffffffu;                            // never an address
    float4 lo = make_float4(0.f, 0.f, 0.f, 0.f), hi = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float kk = kk0 + (float)i;
        const float tx = fmaf(es.x, kk, ea.x), ty = fmaf(es.y, kk, ea.y), tz = fmaf(es.z, kk, ea.z);
        const float rx = __fadd_rd(tx, OAT_MAGIC), ry = __fadd_rd(ty, OAT_MAGIC), rz = __fadd_rd(tz, OAT_MAGIC);
        const unsigned adr = __float_as_uint(rz) * (16u * TT_PZ) + (__float_as_uint(ry) * (16u * TT_PY) + (__float_as_uint(rx) * 16u + Kr));
        lds_records_if_new(lo, hi, adr, prev);
        const float fx = tx - (rx - OAT_MAGIC), fy = ty - (ry - OAT_MAGIC), fz = tz - (rz - OAT_MAGIC);
        const float blo = fmaf(fy, fmaf(fx, lo.w, lo.z), fmaf(fx, lo.y, lo.x));
        const float bhi = fmaf(fy, fmaf(fx, hi.w, hi.z), fmaf(fx, hi.y, hi.x));
        const float v = fmaf(fz, bhi - blo, blo);
        acc[0][i] = fmaf(m0, v, acc[0][i]); acc[1][i] = fmaf(m1, v, acc[1][i]);
        acc[2][i] = fmaf(m2, v, acc[2][i]); acc[3][i] = fmaf(m3, v, acc[3][i]);
    }
}

// ------------------------------------------------------------------------------------------------
// brick load: raw nodes by TMA (or plain loads when the volume's row pitch / address does not fit a tensor map), two rounds of
// 12 node planes through the staging buffer, bilinear plane records into `rec`
// ------------------------------------------------------------------------------------------------
__device__ void load_brick(SmemLayout &S, const OatDev &P, const CUtensorMap *tmap, const float *__restrict__ x, int use_tma,
                           const int (&rlo)[3], unsigned &phase, int tid)
{
    // node (real index) of staging element (sx, sy, sz) of round r: (rlo_x - 2 + sx, rlo_y - 1 + sy, rlo_z - 1 + 12 r + sz)
    for (int r = 0; r < 2; ++r) {
        const int z0 = rlo[2] - 1 + TT_BZ * r;
        if (use_tma) {
            if (tid == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the buffer was last touched by ordinary loads / stores
                mbar_expect_tx(&S.mbar, TT_STAGE_BYTES);
                tma_load_3d(S.u.stage, tmap, &S.mbar, rlo[0] - 2, rlo[1] - 1, z0);   // x start: a multiple of 4 elements (TMA: 16-byte aligned rows)
            }
            mbar_wait(&S.mbar, phase);
            phase ^= 1u;
        } else {
            for (int i = tid; i < TT_BX * TT_BY * TT_BZ; i += TT_THREADS) {
                const int sx = i % TT_BX, sy = (i / TT_BX) % TT_BY, sz = i / (TT_BX * TT_BY);
                const int X = rlo[0] - 2 + sx, Y = rlo[1] - 1 + sy, Z = z0 + sz;
                float v = 0.f;
                if (X >= 0 && X < P.nx && Y >= 0 && Y < P.ny && Z >= 0 && Z < P.nz) v = x[((size_t)Z * P.ny + Y) * P.nx + X];
                S.u.stage[i] = v;
            }
            __syncthreads();
        }
        const int npl = r == 0 ? TT_BZ : TT_NP - TT_BZ;
        if (tid < TT_R * TT_R) {                           // one thread per cell column, all planes of the round
            const int px = tid % TT_R, py = tid / TT_R;
            const float *s = S.u.stage + py * TT_BX + px + 1;
            float4 *dst = S.rec + (TT_BZ * r) * TT_PZ + py * TT_PY + px;
            for (int pl = 0; pl < npl; ++pl, s += TT_BX * TT_BY, dst += TT_PZ) {
                const double v00 = s[0], v10 = s[1], v01 = s[TT_BX], v11 = s[TT_BX + 1];
                const double c1 = v10 - v00, c2 = v01 - v00, c3 = v11 - v01 - c1;
                *dst = make_float4((float)v00, (float)c1, (float)c2, (float)c3);
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// H (projection)
// ------------------------------------------------------------------------------------------------
// Interval of relative azimuths x = phi - phc (|x| <= pi) in which ring (st, ct) at radius s can have a point inside the core:
// per axis a the coordinate is R_a cos(phi - phi0_a) + C_a, so 0 <= coordinate < TT_C holds on two arcs aU <= |phi - phi0_a| <= aL;
// the window [xl, xh] is intersected with both arcs and replaced by the hull of what is left.  Conservative (a superset).
__device__ __forceinline__ void clip_arc(float &xl, float &xh, float c0, float aU, float aL)
{
    // arcs [c0 + aU, c0 + aL] and [c0 - aL, c0 - aU], each also shifted by -/+ 2 pi; c0 in [-pi, pi], window within [-pi, pi]
    float nl = 1e30f, nh = -1e30f;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const float sh = (t & 1) ? ((t & 2) ? 6.2831853f : -6.2831853f) : 0.f;
        const float lo = ((t & 2) ? c0 - aL : c0 + aU) + sh, hi = ((t & 2) ? c0 - aU : c0 + aL) + sh;
        const float il = fmaxf(lo, xl), ih = fminf(hi, xh);
        if (il <= ih) { nl = fminf(nl, il); nh = fmaxf(nh, ih); }
    }
    xl = nl; xh = nh;
}

// H: x -> g, records from the brick.  (A tile-stationary H^T on the same enumeration, with fixed-point node accumulators in
// shared memory, was measured in round 2 -- profiles/r2_tile_bwd.md, DESIGN.md 5.9 -- and is no longer part of the library:
// 2.05x slower than the marching H^T and outside the 1e-4 product tolerance.)
template <bool STATS>
__global__ void __launch_bounds__(TT_THREADS, 1)
oat_tile_kernel(const __grid_constant__ CUtensorMap tmap, const OatDev P, const TileParams T, const float *__restrict__ x,
                double *__restrict__ g, unsigned long long *__restrict__ counter, unsigned long long *__restrict__ stats)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SmemLayout &S = *reinterpret_cast<SmemLayout *>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float stepf = (float)P.step;
    const float s0f = (float)(P.t0 * P.step / P.dt);                     // radius of sample 0 in voxel units
    const unsigned lt_mask = (1u << lane) - 1u;
    float4 *const qa = S.u.q.qa[warp], *const qs = S.u.q.qs[warp];
    unsigned char *const qc = S.qc[warp];
    unsigned *const cq = S.cq[warp];
    double *const s_frame = S.frame[warp];
    float *const s_ff = S.framef[warp];
    const unsigned rec_base = smem_u32(S.rec);
    unsigned phase = 0;
    long long cur_tile = -1;
    unsigned st_cand = 0, st_pre = 0, st_ray = 0, st_chunk = 0;         // STATS: candidates, after the fp32 cull, rays / chunks owned

    if (tid == 0) { mbar_init(&S.mbar, 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
    __syncthreads();

    for (;;) {
        if (tid == 0) S.item = (long long)atomicAdd(counter, 1ULL);
        __syncthreads();
        const long long item = S.item;
        if (item >= T.n_items) break;
        const long long tile = item / T.n_qc;
        const int qc_i = (int)(item % T.n_qc);
        const int tz = (int)(tile / ((long long)T.ntx * T.nty)), ty = (int)((tile / T.ntx) % T.nty), tx = (int)(tile % T.ntx);
        const int clo[3] = {-TT_M + TT_C * tx, -TT_M + TT_C * ty, -TT_M + TT_C * tz};
        const int rlo[3] = {clo[0] - TT_M, clo[1] - TT_M, clo[2] - TT_M};
        if (tile != cur_tile) { load_brick(S, P, &tmap, x, T.use_tma, rlo, phase, tid); cur_tile = tile; }
        if (tid == 0) S.nextq = 0;
        __syncthreads();
        const int q_begin = qc_i * T.nq, q_end = min(P.Q, q_begin + T.nq);

        for (;;) {
            int q = 0;
            if (lane == 0) q = q_begin + atomicAdd(&S.nextq, 1);
            q = __shfl_sync(0xffffffffu, q, 0);
            if (q >= q_end) break;
            __syncwarp();
            if (lane < 12) { const double f = P.frame[(size_t)q * 12 + lane]; s_frame[lane] = f; s_ff[lane] = (float)f; }
            __syncwarp();
            // distance range of the core from the transducer -> sample range -> bands
            float dn2 = 0.f, df2 = 0.f;
            float vb[3];                                   // base' - core lo (fp32: culls only)
            float rho_a[3], phi0_a[3];                     // |(e_x, e_y)_a| and atan2(e_y_a, e_x_a): coordinate a of a ring point is R cos(phi - phi0) + C
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float v = (float)(s_frame[9 + a] - (double)clo[a]);
                vb[a] = v;
                const float dnear = fmaxf(fmaxf(-v, v - (float)TT_C), 0.f);
                const float dfar = fmaxf(fabsf(v), fabsf(v - (float)TT_C));
                dn2 = fmaf(dnear, dnear, dn2); df2 = fmaf(dfar, dfar, df2);
                rho_a[a] = sqrtf(s_ff[a] * s_ff[a] + s_ff[3 + a] * s_ff[3 + a]);
                phi0_a[a] = atan2f(s_ff[3 + a], s_ff[a]);
            }
            const float dmin = sqrtf(dn2), dmax = sqrtf(df2);
            int k_lo = (int)floorf((dmin - s0f) / stepf) - 1, k_hi = (int)ceilf((dmax - s0f) / stepf) + 1;
            if (k_hi < 0 || k_lo > P.K - 1) continue;
            k_lo = max(k_lo, 0); k_hi = min(k_hi, P.K - 1);
            for (int b = k_lo >> 5; b <= (k_hi >> 5); ++b) {
                const OatBand band = P.band[b];
                const int nrq = P.qb_rings[(size_t)q * P.NB + b];
                if (nrq <= 0) continue;
                __syncwarp();
                if (lane == 0) { s_frame[12] = band.s_mid; s_frame[13] = (double)band.s_lo; s_frame[14] = (double)band.s_hi; }
                __syncwarp();
                const OatRing *__restrict__ ring = P.ring + band.ring_ofs;
                const double2 *__restrict__ dir = P.dir + band.dir_ofs;
                // ---- window of rings and azimuths that covers the core's projection: 27 lattice points of the core
                float th, ph, rp;
                {
                    const int li = lane < 27 ? lane : 13;
                    const float px = (float)(TT_C / 2) * (float)(li % 3) - vb[0], py = (float)(TT_C / 2) * (float)((li / 3) % 3) - vb[1],
                                pz = (float)(TT_C / 2) * (float)(li / 9) - vb[2];
                    const float X = px * s_ff[0] + py * s_ff[1] + pz * s_ff[2], Y = px * s_ff[3] + py * s_ff[4] + pz * s_ff[5],
                                Z = px * s_ff[6] + py * s_ff[7] + pz * s_ff[8];
                    rp = sqrtf(X * X + Y * Y);
                    th = atan2f(rp, Z);
                    ph = atan2f(Y, X);
                }
                const float phc = __shfl_sync(0xffffffffu, ph, 13), rpc = __shfl_sync(0xffffffffu, rp, 13);
                const float dth = (float)band.dtheta;
                const float thmin = warp_min(th), thmax = warp_max(th), rpmin = warp_min(rp);
                // theta is largest at a corner, but its minimum may lie inside a face or an edge: the distance to the axis is convex
                // with curvature <= 1 / distance, so between lattice points (at most 5.66 cells away) it undercuts them by < 16 / r
                const float slack = rpmin > 6.f ? 16.f / rpmin + 0.5f : 1e30f;               // cells
                int i0 = (int)floorf((thmin - slack / fmaxf(dmin, 1.f)) / dth) - 1, i1 = (int)ceilf(thmax / dth) + 1;   // ring numbers i = 1, 2, ..
                if (!(slack < 1e29f)) i0 = 1;
                const bool nearq = dmin < 2.f * (float)TT_C;                                 // the transducer sits in or next to the core: no window
                if (nearq) { i0 = 1; i1 = nrq; }
                i0 = max(i0, 1); i1 = min(i1, nrq);
                if (i0 > i1) continue;
                const bool full = nearq || rpc < 0.5f * 1.7320508f * (float)TT_C + 2.f;      // the axis passes through or near the core
                float dl = ph - phc;
                dl = dl > 3.14159265f ? dl - 6.2831853f : (dl < -3.14159265f ? dl + 6.2831853f : dl);
                const float dlmin = warp_min(dl), dlmax = warp_max(dl);
                const float sa = (float)band.s_mid - 15.5f * stepf, sb = sa + 24.f * stepf;   // radii of the first samples of chunks 0 and 3
                const int nch = min(4, (band.nk + 7) >> 3);                                   // chunks of this band
                float acc[4][8];                                                              // [chunk index][step]: sample 8 c + i of the band
#pragma unroll
                for (int c = 0; c < 4; ++c)
#pragma unroll
                    for (int i = 0; i < 8; ++i) acc[c][i] = 0.f;
                int head = 0, cnt = 0;                                                        // chunk queue
                int chead = 0, ccnt = 0;                                                      // candidate queue
                // ring block (32 rings, lane l keeps ring ib + l) and the rays of the last phase 2 (their chunks are appended one index at a time)
                int ib = i0 - 32, nb = 0, n_rows = 0, row = 0, W = 32, wsh = 5, nseg = 1;
                int rN = 1, rcum = 0, rn = 0, rjl = 0;
                float rst = 0.f, rctf = 1.f, rom = 0.f, rdphi = 0.f;
                double rct = 1.0;
                Ray e;
                e.ax = e.ay = e.az = 0.f; e.sx = e.sy = e.sz = 0.f; e.ix = e.iy = e.iz = 0;
                unsigned own = 0, Kc = 0;
                float om = 0.f;
                int pend = 4;
                bool all_done = false;
#pragma unroll 1
                for (;;) {
                    if (cnt >= 32 || (all_done && cnt > 0)) {
                        march_group_fwd(qa, qs, qc, head, cnt, acc, lane, rec_base);
                        continue;
                    }
                    if (all_done) break;
                    if (pend < 4) {
                        // ------------------------------------------------------------ append chunk `pend` of the current rays
                        const bool mine = (own >> pend) & 1u;
                        const unsigned m = __ballot_sync(0xffffffffu, mine);
                        if (mine) {
                            const int slot = (head + cnt + __popc(m & lt_mask)) & (TT_QN - 1);
                            qa[slot] = make_float4(e.ax, e.ay, e.az, om);
                            qs[slot] = make_float4(e.sx, e.sy, e.sz, __uint_as_float(Kc));
                            qc[slot] = (unsigned char)pend;
                        }
                        cnt += __popc(m);
                        ++pend;
                        __syncwarp();
                        continue;
                    }
                    const bool rows_done = row >= n_rows;
                    if (ccnt >= 32 || (rows_done && ccnt > 0)) {
                        // ------------------------------------------------------------ phase 2: 32 candidates -> fp64 anchors -> owned chunks
                        const int n2 = min(ccnt, 32);
                        bool ok = lane < n2;
                        const unsigned ce = ok ? cq[(chead + lane) & (TT_QN - 1)] : 0u;
                        __syncwarp();
                        chead = (chead + n2) & (TT_QN - 1);
                        ccnt -= n2;
                        const int src = (int)(ce >> 27);
                        const double ct = __shfl_sync(0xffffffffu, rct, src);
                        om = __shfl_sync(0xffffffffu, rom, src);
                        double2 d = make_double2(0.0, 0.0);
                        if (ok) d = dir[ce & 0x7ffffffu];
                        own = 0;
                        ok = make_ray(P, d, ct, stepf, s_frame, e) && ok;
                        if (ok) {
#pragma unroll
                            for (int c = 0; c < 4; ++c) {
                                const float kk = 8.f * (float)c - 15.5f;
                                const float t0 = fmaf(e.sx, kk, e.ax), t1 = fmaf(e.sy, kk, e.ay), t2 = fmaf(e.sz, kk, e.az);
                                const int c0 = e.ix + (int)floorf(t0) - clo[0], c1 = e.iy + (int)floorf(t1) - clo[1],
                                          c2 = e.iz + (int)floorf(t2) - clo[2];
                                if (c < nch && (unsigned)c0 < (unsigned)TT_C && (unsigned)c1 < (unsigned)TT_C && (unsigned)c2 < (unsigned)TT_C)
                                    own |= 1u << c;
                            }
                        }
                        if (STATS) { st_ray += own ? 1 : 0; st_chunk += __popc(own); }
                        Kc = rec_base + 16u * (((unsigned)(e.ix - rlo[0]) - OAT_MAGIC_BITS) + (unsigned)TT_PY * ((unsigned)(e.iy - rlo[1]) - OAT_MAGIC_BITS)
                                               + (unsigned)TT_PZ * ((unsigned)(e.iz - rlo[2]) - OAT_MAGIC_BITS));
                        if (__any_sync(0xffffffffu, own != 0u)) pend = 0;
                        continue;
                    }
                    if (!rows_done) {
                        // ------------------------------------------------------------ phase 1 (fp32, no memory): candidate -> cull against the core
                        const int rr = nseg == 1 ? row : row / nseg, sg = nseg == 1 ? 0 : row % nseg;
                        const int rl = (rr << (5 - wsh)) + (lane >> wsh);                     // ring slot of this lane's candidate
                        const int jj = sg * 32 + (lane & (W - 1));
                        const int src = rl & 31;
                        const int N = __shfl_sync(0xffffffffu, rN, src), n = __shfl_sync(0xffffffffu, rn, src);
                        const int jl = __shfl_sync(0xffffffffu, rjl, src), cum = __shfl_sync(0xffffffffu, rcum, src);
                        const float st = __shfl_sync(0xffffffffu, rst, src), ctf = __shfl_sync(0xffffffffu, rctf, src);
                        const float dphi = __shfl_sync(0xffffffffu, rdphi, src);
                        bool ok = rl < nb && jj < n;
                        int j = jl + jj;
                        j = j >= N ? j - N : j;
                        if (STATS) st_cand += ok ? 1 : 0;
                        float sn, cs;
                        __sincosf((float)j * dphi, &sn, &cs);
                        const float dx = st * cs, dy = st * sn;
#pragma unroll
                        for (int a = 0; a < 3; ++a) {
                            const float ua = dx * s_ff[a] + dy * s_ff[3 + a] + ctf * s_ff[6 + a];
                            const float p0 = fmaf(sa, ua, vb[a]), p1 = fmaf(sb, ua, vb[a]);
                            ok = ok && (fmaxf(p0, p1) >= -0.05f) && (fminf(p0, p1) <= (float)TT_C + 0.05f);
                        }
                        if (STATS) st_pre += ok ? 1 : 0;
                        const unsigned m = __ballot_sync(0xffffffffu, ok);
                        if (ok) {
                            cq[(chead + ccnt + __popc(m & lt_mask)) & (TT_QN - 1)] = ((unsigned)src << 27) | (unsigned)(cum + j);
                            prefetch_l1(dir + (cum + j));
                        }
                        ccnt += __popc(m);
                        ++row;
                        __syncwarp();
                        continue;
                    }
                    // ---------------------------------------------------------------- next block of 32 rings
                    ib += 32;
                    if (ib > i1) { all_done = true; continue; }
                    rN = 1; rcum = 0; rn = 0; rjl = 0; rst = 0.f; rctf = 1.f; rom = 0.f; rdphi = 0.f; rct = 1.0;
                    if (ib + lane <= i1) {
                        const OatRing *rp_ = ring + (ib + lane - 1);
                        rN = rp_->N; rcum = rp_->cum; rct = rp_->ct; rst = (float)rp_->st; rom = rp_->omega;
                        rctf = (float)rct;
                        rdphi = 6.2831853f / (float)rN;
                        const float sc = (float)rN * 0.15915494f;                             // N / (2 pi)
                        rn = rN;
                        if (!full) {
                            // azimuth interval of this ring: hull over the chunk radii of (window of the core's corners) x (arcs per axis)
                            float XL = 1e30f, XH = -1e30f;
#pragma unroll 1
                            for (int c = 0; c < nch; ++c) {
                                const float s = fmaf(8.f * (float)c, stepf, sa);
                                float xl = dlmin - 2e-3f, xh = dlmax + 2e-3f;
#pragma unroll
                                for (int a = 0; a < 3; ++a) {
                                    const float R = s * rst * rho_a[a];
                                    const float C = fmaf(s * rctf, s_ff[6 + a], vb[a]);
                                    const float L = -0.1f - C, U = (float)TT_C + 0.1f - C;
                                    if (R < 1e-4f) { if (!(L <= 0.f && 0.f <= U)) { xl = 1e30f; xh = -1e30f; } continue; }
                                    const float uL = L / R, uU = U / R;
                                    if (uL > 1.f || uU < -1.f) { xl = 1e30f; xh = -1e30f; continue; }
                                    const float aL = uL <= -1.f ? 3.1415927f : acosf(uL), aU = uU >= 1.f ? 0.f : acosf(uU);
                                    float c0 = phi0_a[a] - phc;
                                    c0 = c0 > 3.14159265f ? c0 - 6.2831853f : (c0 < -3.14159265f ? c0 + 6.2831853f : c0);
                                    clip_arc(xl, xh, c0, aU - 2e-3f, aL + 2e-3f);
                                }
                                if (xl <= xh) { XL = fminf(XL, xl); XH = fmaxf(XH, xh); }
                            }
                            if (XL <= XH) {
                                rjl = (int)ceilf((phc + XL) * sc) - 1;
                                rn = min(rN, (int)floorf((phc + XH) * sc) - rjl + 2);
                                rjl %= rN; if (rjl < 0) rjl += rN;
                            } else rn = 0;
                        }
                    }
                    int nmax = rn;
#pragma unroll
                    for (int s = 16; s >= 1; s >>= 1) nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, s));
                    wsh = nmax <= 8 ? 3 : nmax <= 16 ? 4 : 5;                                 // lanes per ring = 1 << wsh
                    W = 1 << wsh;
                    nseg = (nmax + 31) / 32;                                                  // rows per ring when a ring is wider than 32
                    nb = min(32, i1 - ib + 1);
                    n_rows = nmax == 0 ? 0 : ((nb + (32 >> wsh) - 1) >> (5 - wsh)) * nseg;
                    row = 0;
                }
                // S5: sum the accumulators over the lanes (lane l collects sample l of the band), one fp64 atomic per time sample
                float accK = 0.f;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float r = warp_transpose_sum8(acc[c], lane);
                    if ((lane >> 3) == c) accK = r;
                }
                const int k = band.k0 + lane;
                const double rho = P.c * (P.t0 + (double)k * P.dt);
                if (lane < band.nk && rho > 0.0 && accK != 0.f) atomicAdd(&g[(size_t)q * P.K + k], rho * rho * (double)accK);
            }
        }
        // all warps meet at the barrier at the top of the loop before the brick or the staging buffer is touched again
    }
    if (STATS) {
        atomicAdd(&stats[0], (unsigned long long)st_cand); atomicAdd(&stats[1], (unsigned long long)st_pre);
        atomicAdd(&stats[2], (unsigned long long)st_ray); atomicAdd(&stats[3], (unsigned long long)st_chunk);
    }
}

// step A4 (Eq. 3 L63 / Eq. 13): y_k = kappa (g_{k+1}/t_{k+1} - g_{k-1}/t_{k-1}) / (2 dt), zero extension (reading G8)
__global__ void oat_tile_diff_kernel(const OatDev P, const double *__restrict__ g, float *__restrict__ y)
{
    const long long n = (long long)P.Q * P.K;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int k = (int)(i % P.K);
        double sp = 0.0, sm = 0.0;
        if (k + 1 < P.K) { const double t = P.t0 + (double)(k + 1) * P.dt; if (t > 0.0) sp = g[i + 1] / t; }
        if (k - 1 >= 0) { const double t = P.t0 + (double)(k - 1) * P.dt; if (t > 0.0) sm = g[i - 1] / t; }
        y[i] = (float)(P.kappa * (sp - sm) / (2.0 * P.dt));
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess && qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

}  // namespace

bool oat_tile_supported(const OatDev &P)
{
    return P.B == 32 && P.dir != nullptr && 7.0 * P.step < (double)TT_M && P.Q > 0 && P.max_band_dirs < (1LL << 27);
}

cudaError_t oat_launch_tile_fwd(const OatDev &P, const float *x, double *g, float *y, unsigned long long *counter,
                                unsigned long long *stats, int nq_per_item, int allow_tma, cudaStream_t st)
{
    TileParams T;
    T.ntx = (P.nx + 1 + 2 * TT_M + TT_C - 1) / TT_C;
    T.nty = (P.ny + 1 + 2 * TT_M + TT_C - 1) / TT_C;
    T.ntz = (P.nz + 1 + 2 * TT_M + TT_C - 1) / TT_C;
    T.nq = nq_per_item > 0 ? nq_per_item : 1024;
    T.n_qc = (P.Q + T.nq - 1) / T.nq;
    T.n_items = (long long)T.ntx * T.nty * T.ntz * T.n_qc;
    T.use_tma = 0;
    CUtensorMap map;
    memset(&map, 0, sizeof(map));
    EncodeTiledFn enc = encode_tiled();
    if (allow_tma && enc && (P.nx % 4) == 0 && ((uintptr_t)x % 16) == 0 && P.nx >= TT_BX && P.ny >= TT_BY && P.nz >= TT_BZ) {
        const cuuint64_t dims[3] = {(cuuint64_t)P.nx, (cuuint64_t)P.ny, (cuuint64_t)P.nz};
        const cuuint64_t strides[2] = {(cuuint64_t)P.nx * 4, (cuuint64_t)P.nx * P.ny * 4};
        const cuuint32_t box[3] = {TT_BX, TT_BY, TT_BZ};
        const cuuint32_t es[3] = {1, 1, 1};
        if (enc(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)x, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS)
            T.use_tma = 1;
    }
    static bool attr_set[64] = {false};
    int dev = 0;
    cudaGetDevice(&dev);
    const int smem = (int)sizeof(SmemLayout);
    if (dev < 0 || dev >= 64 || !attr_set[dev]) {
        cudaError_t e = cudaFuncSetAttribute(oat_tile_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(oat_tile_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_set[dev] = true;
    }
    int n_sm = 148;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    const long long grid = T.n_items < n_sm ? T.n_items : n_sm;
    if (stats) oat_tile_kernel<true><<<(unsigned)grid, TT_THREADS, smem, st>>>(map, P, T, x, g, counter, stats);
    else oat_tile_kernel<false><<<(unsigned)grid, TT_THREADS, smem, st>>>(map, P, T, x, g, counter, stats);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const long long n = (long long)P.Q * P.K;
    long long gsz = (n + 255) / 256;
    if (gsz > 148LL * 16) gsz = 148LL * 16;
    oat_tile_diff_kernel<<<(unsigned)gsz, 256, 0, st>>>(P, g, y);
    return cudaGetLastError();
}
