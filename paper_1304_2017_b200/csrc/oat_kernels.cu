// CUDA kernels of liboat.so for sm_100a (B200).  No tensor cores: H is a gather /
// interpolate / accumulate over sphere-surface samples, not a dense contraction.
//
// Ray kernel (variant 0, "ray lanes").  A work item is a chunk of
// candidate directions of one (transducer q, band b of B <= 32 time samples).  The block
//   1. BUILDS in shared memory the list of directions (ring i, azimuth j) of that chunk whose
//      ray segment [rho_first, rho_last] can meet the zero-padded node box: a cheap fp32
//      pre-test, then for the survivors the direction u (S3) and the ray's anchor point
//      base' + s_mid*u in fp64, split into an integer node offset and a fraction in [-0.5, 0.5];
//   2. CONSUMES the list: warp = one direction, lane = one time sample k of the band, so the
//      32 lanes step along one ray (c*dt/ds voxels apart) and a warp-wide corner load touches
//      only a few cache lines.  Sample position = fma(delta_k, u, anchor_frac): one fp32 rounding
//      at |t| < ~6 voxels, i.e. ~3e-7 voxel -- the fp64-anchored form is what keeps H within
//      1e-4 of the fp64 oracle after the time difference amplifies errors ~30x.
// The same list and the same per-lane position/weight code serve H (gather), H^T (scatter) and
// the sample counter, so the three visit exactly the same samples with the same weights
// (Eq. 12 vs Eq. 23; Alg. 4 vs Alg. 6).
#include "oat_internal.h"

#include <math.h>

#include <cub/device/device_radix_sort.cuh>

namespace {

#define OAT_MAGIC_BITS_C 0x4B400000   // bit pattern of 1.5 * 2^23 (OAT_MAGIC below)
struct __align__(16) Entry {
    float4 a;   // anchor fraction (x,y,z) in [-0.5,0.5], omega
    float4 u;   // direction (x,y,z) in voxel axes, unused
    int4 i;     // anchor integer node offset in the padded volume (x,y,z), unused
};

// 32-byte list entry of the marching kernels: the three integer anchor offsets (each in [-OAT_PB, 1023 - OAT_PB]:
// checked at variant selection) packed into the bit pattern of u.w.  A third less shared memory per block than
// Entry: what is not carved out for shared memory is L1, and the rate at which L1 serves the scattered record loads
// of H falls with its size (micro-benchmark in profiles/r1h_*).
#define OAT_PB 128
struct __align__(16) PEntry {
    float4 a;   // anchor fraction (x,y,z), omega
    float4 u;   // direction (x,y,z), packed anchor node offsets
};

__device__ __forceinline__ PEntry pack_entry(const Entry &e)
{
    PEntry p;
    p.a = e.a;
    const unsigned pk = (unsigned)(e.i.x + OAT_MAGIC_BITS_C + OAT_PB) | ((unsigned)(e.i.y + OAT_MAGIC_BITS_C + OAT_PB) << 10) |
                        ((unsigned)(e.i.z + OAT_MAGIC_BITS_C + OAT_PB) << 20);
    p.u = make_float4(e.u.x, e.u.y, e.u.z, __uint_as_float(pk));
    return p;
}

__device__ __forceinline__ Entry unpack_entry(const PEntry &p)
{
    Entry e;
    e.a = p.a;
    e.u = make_float4(p.u.x, p.u.y, p.u.z, 0.f);
    const unsigned pk = __float_as_uint(p.u.w);
    e.i = make_int4((int)(pk & 1023u) - (OAT_MAGIC_BITS_C + OAT_PB), (int)((pk >> 10) & 1023u) - (OAT_MAGIC_BITS_C + OAT_PB),
                    (int)((pk >> 20) & 1023u) - (OAT_MAGIC_BITS_C + OAT_PB), 0);
    return e;
}

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// per-lane sample of one list entry: padded cell index and fractions; returns in-box flag
struct Sample {
    int ix, iy, iz;
    float fx, fy, fz;
};

// floor() without the quarter-rate conversion pipe: adding 1.5*2^23 with round-toward-minus-infinity
// leaves floor(t) in the low mantissa bits (|t| < 2^22), so the integer cell index is one integer add
// away from the float's bit pattern and floor(t) as a float is one exact subtraction away.
#define OAT_MAGIC 12582912.0f
#define OAT_MAGIC_BITS 0x4B400000

__device__ __forceinline__ bool lane_sample(const OatDev &P, const Entry &e, float delta, Sample &s)
{
    const float tx = fmaf(delta, e.u.x, e.a.x);
    const float ty = fmaf(delta, e.u.y, e.a.y);
    const float tz = fmaf(delta, e.u.z, e.a.z);
    const float rx = __fadd_rd(tx, OAT_MAGIC), ry = __fadd_rd(ty, OAT_MAGIC), rz = __fadd_rd(tz, OAT_MAGIC);
    s.ix = __float_as_int(rx) + e.i.x;                   // e.i.* carry the -OAT_MAGIC_BITS bias
    s.iy = __float_as_int(ry) + e.i.y;
    s.iz = __float_as_int(rz) + e.i.z;
    s.fx = tx - (rx - OAT_MAGIC);
    s.fy = ty - (ry - OAT_MAGIC);
    s.fz = tz - (rz - OAT_MAGIC);
    // padded cell n' in [0, N] <=> xi in [-1, N): the sample touches at least one existing node (S4)
    return ((unsigned)s.ix <= (unsigned)P.nx) & ((unsigned)s.iy <= (unsigned)P.ny) & ((unsigned)s.iz <= (unsigned)P.nz);
}

__device__ __forceinline__ void red_add_v4(float4 *addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// index of the quad that holds the in-plane corners of padded cell (ix, iy) in plane iz
__device__ __forceinline__ unsigned quad_index(const OatDev &P, int ix, int iy, int iz)
{
    const int par = (ix & 1) | ((iy & 1) << 1);          // 4*pz*qplane < 2^31 is checked at create
    return (unsigned)(((par * P.pz + iz) * P.qy + (iy >> 1)) * P.qx + (ix >> 1));
}

// the 8 corner values of the sample's cell (v[cz*4 + cy*2 + cx]); lanes that are not in the box read
// cell 0 (valid memory) so that the loads of several list entries can be issued back to back
template <int VAR>
__device__ __forceinline__ void fetch8(const OatDev &P, const float *__restrict__ xpad, const Sample &s, bool in, float v[8])
{
    const int ix = in ? s.ix : 0, iy = in ? s.iy : 0, iz = in ? s.iz : 0;
    if (VAR == 0) {                                       // 8 scalar loads from the padded linear volume
        const float *p = xpad + (unsigned)((iz * P.py + iy) * P.px + ix);
        v[0] = __ldg(p); v[1] = __ldg(p + 1);
        v[2] = __ldg(p + P.px); v[3] = __ldg(p + P.px + 1);
        const float *p1 = p + P.pxy;
        v[4] = __ldg(p1); v[5] = __ldg(p1 + 1);
        v[6] = __ldg(p1 + P.px); v[7] = __ldg(p1 + P.px + 1);
    } else if (VAR == 3) {                                // ONE 256-bit load from the parity-shifted octet arrays
        const int par = (ix & 1) | ((iy & 1) << 1) | ((iz & 1) << 2);
        const unsigned oi = (unsigned)(((par * P.oz + (iz >> 1)) * P.qy + (iy >> 1)) * P.qx + (ix >> 1));
        const float *op = xpad + (size_t)oi * 8;
        asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                     : "l"(op));
    } else if (VAR == 2) {                                // 2 x LDG.128 from the parity-shifted quad arrays
        const float4 *qp = reinterpret_cast<const float4 *>(xpad) + quad_index(P, ix, iy, iz);
        const float4 lo = __ldg(qp), hi = __ldg(qp + P.qplane);
        v[0] = lo.x; v[1] = lo.y; v[2] = lo.z; v[3] = lo.w;
        v[4] = hi.x; v[5] = hi.y; v[6] = hi.z; v[7] = hi.w;
    } else {                                              // 2 texture gathers (tld4) from the slice atlas
        const int z1 = iz + 1;
        const float tx = (float)ix + 1.0f, ty = (float)iy + 1.0f;   // between texel centres: exact 2x2 footprint
        const float ax0 = (float)((iz & P.atlas_mask) * P.px), ay0 = (float)((iz >> P.atlas_shift) * P.py);
        const float ax1 = (float)((z1 & P.atlas_mask) * P.px), ay1 = (float)((z1 >> P.atlas_shift) * P.py);
        const float4 lo = tex2Dgather<float4>(P.tex, tx + ax0, ty + ay0, 0);
        const float4 hi = tex2Dgather<float4>(P.tex, tx + ax1, ty + ay1, 0);
        // gather order: x = (i, j+1), y = (i+1, j+1), z = (i+1, j), w = (i, j)
        v[0] = lo.w; v[1] = lo.z; v[2] = lo.x; v[3] = lo.y;
        v[4] = hi.w; v[5] = hi.z; v[6] = hi.x; v[7] = hi.y;
    }
}

#define OAT_U 4    // list entries in flight per warp (independent dependency chains)

// Per-lane constants of one (transducer q, band): lane = time sample k of the band.
struct LaneCtx {
    int k;
    double rho;
    bool active;
    float delta;   // radial offset of sample k from the band anchor, in voxels
    float coef;    // MODE 1: g'_k * rho_k^2  (S7, S8)
};

template <int MODE>
__device__ __forceinline__ LaneCtx lane_setup(const OatDev &P, const OatBand &band, int q, int lane, const float *__restrict__ y)
{
    LaneCtx c;
    c.k = band.k0 + lane;
    const double tk = P.t0 + (double)c.k * P.dt;
    c.rho = P.c * tk;
    c.active = (lane < band.nk) && (c.rho > 0.0);
    c.delta = (float)(((double)lane - 0.5 * (double)(P.B - 1)) * P.step);
    c.coef = 0.f;
    if (MODE == 1 && c.active) {
        const float ym = (c.k - 1 >= 0) ? y[(size_t)q * P.K + c.k - 1] : 0.f;
        const float yp = (c.k + 1 < P.K) ? y[(size_t)q * P.K + c.k + 1] : 0.f;
        const double sp = P.kappa * ((double)ym - (double)yp) / (2.0 * P.dt);   // Eq. 22
        c.coef = (float)(sp / tk * c.rho * c.rho);
    }
    return c;
}

// Direction (S3) of ring R, azimuth j in the frame of the transducer, and the ray's anchor point
// base' + s_mid*u, all in fp64; returns false when the bounding box of the ray segment
// [s_lo, s_hi] cannot meet the padded node box.
__device__ __forceinline__ bool make_entry(const OatDev &P, const OatBand &band, const OatRing &R, int j,
                                           const double *s_frame, Entry &e)
{
    double sd, cd;
    sincospi(2.0 * (double)j / (double)R.N, &sd, &cd);
    const double dlx = R.st * cd, dly = R.st * sd, dlz = R.ct;
    float uu[3], af[3];
    int ai[3];
    bool hit = true;
    const float lim[3] = {(float)P.nx + 1.01f, (float)P.ny + 1.01f, (float)P.nz + 1.01f};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double ua = dlx * s_frame[a] + dly * s_frame[3 + a] + dlz * s_frame[6 + a];
        const double an = s_frame[9 + a] + band.s_mid * ua;
        const double ar = rint(an);
        uu[a] = (float)ua;
        af[a] = (float)(an - ar);
        ai[a] = (int)ar;
        const float p0 = (float)(s_frame[9 + a] + (double)band.s_lo * ua);
        const float p1 = (float)(s_frame[9 + a] + (double)band.s_hi * ua);
        hit = hit && (fmaxf(p0, p1) >= -0.01f) && (fminf(p0, p1) <= lim[a]);
    }
    e.a = make_float4(af[0], af[1], af[2], R.omega);
    e.u = make_float4(uu[0], uu[1], uu[2], 0.f);
    e.i = make_int4(ai[0] - OAT_MAGIC_BITS, ai[1] - OAT_MAGIC_BITS, ai[2] - OAT_MAGIC_BITS, 0);
    return hit;
}

// CONSUME: one warp per list entry (one ray), lane = time sample; OAT_U entries in flight.
template <int MODE, int VAR>
__device__ __forceinline__ void consume_list(const OatDev &P, const Entry *__restrict__ list, int n_list, int warp, int lane,
                                             const LaneCtx &L, const float *__restrict__ xpad, float *__restrict__ xacc,
                                             float &acc, unsigned &cnt)
{
    const float delta = L.delta, coef = L.coef;
    const bool active = L.active;
    for (int e0 = warp; e0 < n_list; e0 += OAT_NW * OAT_U) {
        Sample s[OAT_U];
        bool in[OAT_U];
        float om[OAT_U];
#pragma unroll
        for (int u = 0; u < OAT_U; ++u) {
            const int ei = e0 + u * OAT_NW;
            const bool valid = ei < n_list;
            const Entry e = list[valid ? ei : e0];
            in[u] = lane_sample(P, e, delta, s[u]) && active && valid;
            om[u] = e.a.w;
        }
        if (MODE == 2) {
#pragma unroll
            for (int u = 0; u < OAT_U; ++u) cnt += in[u] ? 1u : 0u;
        } else if (MODE == 0) {
            float v[OAT_U][8];
#pragma unroll
            for (int u = 0; u < OAT_U; ++u) fetch8<VAR>(P, xpad, s[u], in[u], v[u]);
#pragma unroll
            for (int u = 0; u < OAT_U; ++u) {
                const float a00 = fmaf(s[u].fx, v[u][1] - v[u][0], v[u][0]);
                const float a10 = fmaf(s[u].fx, v[u][3] - v[u][2], v[u][2]);
                const float a01 = fmaf(s[u].fx, v[u][5] - v[u][4], v[u][4]);
                const float a11 = fmaf(s[u].fx, v[u][7] - v[u][6], v[u][6]);
                const float b0 = fmaf(s[u].fy, a10 - a00, a00);
                const float b1 = fmaf(s[u].fy, a11 - a01, a01);
                acc = fmaf(in[u] ? om[u] : 0.f, fmaf(s[u].fz, b1 - b0, b0), acc);
            }
        } else {
#pragma unroll
            for (int u = 0; u < OAT_U; ++u) {
                const unsigned idx = (VAR == 2) ? quad_index(P, s[u].ix, s[u].iy, s[u].iz)
                                                : (unsigned)((s[u].iz * P.py + s[u].iy) * P.px + s[u].ix);
                const float cw = in[u] ? coef * om[u] : 0.f;
                const float wz1 = s[u].fz * cw, wz0 = cw - wz1;
                const float gx = 1.f - s[u].fx, gy = 1.f - s[u].fy;
                const float w00 = gx * gy, w10 = s[u].fx * gy, w01 = gx * s[u].fy, w11 = s[u].fx * s[u].fy;
                float w[8] = {w00 * wz0, w10 * wz0, w01 * wz0, w11 * wz0, w00 * wz1, w10 * wz1, w01 * wz1, w11 * wz1};
                bool writer = in[u];
                if (VAR >= 1) {
                    // Lanes step along one ray, so lanes that fall into the same cell are CONSECUTIVE:
                    // sum each run into its first lane (segmented suffix sum by shuffles) and let only
                    // run heads issue the atomics (~3x fewer L2 atomic operations).
                    const unsigned cell = in[u] ? idx : (0xfffffff0u - (unsigned)lane);
                    const unsigned prev = __shfl_up_sync(0xffffffffu, cell, 1);
                    const bool head = (lane == 0) || (cell != prev);
                    const unsigned heads = __ballot_sync(0xffffffffu, head);
                    const unsigned above = (lane == 31) ? 0u : (heads & ~((2u << lane) - 1u));
                    const int run_end = above ? (__ffs(above) - 2) : 31;
                    const unsigned maxrun = __reduce_max_sync(0xffffffffu, (head && in[u]) ? (unsigned)(run_end - lane + 1) : 0u);
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        if (maxrun > (unsigned)d) {                    // warp-uniform
                            const float keep = (lane + d <= run_end) ? 1.f : 0.f;
#pragma unroll
                            for (int c = 0; c < 8; ++c) w[c] = fmaf(keep, __shfl_down_sync(0xffffffffu, w[c], d), w[c]);
                        }
                    }
                    writer = in[u] && head;
                }
                if (VAR == 2) {
                    // one aligned 16-byte vector reduction per plane: 2 L2 sector operations per run
                    if (writer) {
                        float4 *qp = reinterpret_cast<float4 *>(xacc) + idx;
                        red_add_v4(qp, w[0], w[1], w[2], w[3]);
                        red_add_v4(qp + P.qplane, w[4], w[5], w[6], w[7]);
                    }
                } else if (writer) {
                    float *p = xacc + idx;
                    atomicAdd(p, w[0]);
                    atomicAdd(p + 1, w[1]);
                    atomicAdd(p + P.px, w[2]);
                    atomicAdd(p + P.px + 1, w[3]);
                    float *p1 = p + P.pxy;
                    atomicAdd(p1, w[4]);
                    atomicAdd(p1 + 1, w[5]);
                    atomicAdd(p1 + P.px, w[6]);
                    atomicAdd(p1 + P.px + 1, w[7]);
                }
            }
        }
    }
}

// CONSUME for H^T, "marching" form (backproject variant 3): one THREAD per ray, stepping through the
// band's time samples in order.  Consecutive samples of a ray that fall in the same cell are summed in
// registers and flushed with two 16-byte vector reductions when the ray leaves the cell -- the same
// run-merging as variant 2 but without any shuffle.  Positions, cells and weights come from the same
// lane_sample() as in H, with the same per-sample delta (table s_delta), so the sample set is identical.
__device__ __forceinline__ void consume_march(const OatDev &P, const Entry *__restrict__ list, int n_list, int tid, int nk,
                                              const float *__restrict__ s_delta, const float *__restrict__ s_coef,
                                              float *__restrict__ xacc)
{
    float4 *__restrict__ quads = reinterpret_cast<float4 *>(xacc);
    for (int ei = tid; ei < n_list; ei += OAT_NT) {
        const Entry e = list[ei];
        unsigned cur = 0xffffffffu;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f, a5 = 0.f, a6 = 0.f, a7 = 0.f;
#pragma unroll 2
        for (int k = 0; k < nk; ++k) {
            const float cw0 = s_coef[k];
            Sample s;
            const bool in = lane_sample(P, e, s_delta[k], s) && (cw0 != 0.f);
            const unsigned cell = in ? quad_index(P, s.ix, s.iy, s.iz) : 0xffffffffu;
            if (cell != cur) {
                if (cur != 0xffffffffu) {
                    red_add_v4(quads + cur, a0, a1, a2, a3);
                    red_add_v4(quads + cur + P.qplane, a4, a5, a6, a7);
                }
                a0 = a1 = a2 = a3 = a4 = a5 = a6 = a7 = 0.f;
                cur = cell;
            }
            if (in) {
                const float cw = cw0 * e.a.w;
                const float wz1 = s.fz * cw, wz0 = cw - wz1;
                const float gx = 1.f - s.fx, gy = 1.f - s.fy;
                const float w00 = gx * gy, w10 = s.fx * gy, w01 = gx * s.fy, w11 = s.fx * s.fy;
                a0 = fmaf(w00, wz0, a0); a1 = fmaf(w10, wz0, a1); a2 = fmaf(w01, wz0, a2); a3 = fmaf(w11, wz0, a3);
                a4 = fmaf(w00, wz1, a4); a5 = fmaf(w10, wz1, a5); a6 = fmaf(w01, wz1, a6); a7 = fmaf(w11, wz1, a7);
            }
        }
        if (cur != 0xffffffffu) {
            red_add_v4(quads + cur, a0, a1, a2, a3);
            red_add_v4(quads + cur + P.qplane, a4, a5, a6, a7);
        }
    }
}

// EPILOGUE of one work item: cross-warp combine in fp64 and one fp64 atomic per time sample (S5)
template <int MODE>
__device__ __forceinline__ void item_epilogue(const OatDev &P, int q, const LaneCtx &L, float acc, unsigned cnt, int warp, int lane,
                                              float (*s_red)[32], double *__restrict__ g, unsigned long long *__restrict__ counter)
{
    if (MODE == 0) {
        s_red[warp][lane] = acc;
        __syncthreads();
        if (warp == 0) {
            double sum = 0.0;
#pragma unroll
            for (int w = 0; w < OAT_NW; ++w) sum += (double)s_red[w][lane];
            if (L.active && sum != 0.0) atomicAdd(&g[(size_t)q * P.K + L.k], L.rho * L.rho * sum);
        }
    } else if (MODE == 2) {
        const double tot = warp_sum((double)cnt);
        if (lane == 0 && tot > 0) atomicAdd(counter, (unsigned long long)tot);
    }
}

// ------------------------------------------------------------------------------------------------
// Schedule 0: work item = chunk of OAT_CH candidate directions (ring-major) of one (q, band)
// ------------------------------------------------------------------------------------------------
template <int MODE, int VAR>
__global__ void __launch_bounds__(OAT_NT, 2)
oat_ray_kernel(const OatDev P, const float *__restrict__ xpad, float *__restrict__ xacc,
               const float *__restrict__ y, double *__restrict__ g, unsigned long long *__restrict__ counter)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Entry *list = reinterpret_cast<Entry *>(smem_raw);
    __shared__ double s_frame[12];
    __shared__ float s_framef[12];
    __shared__ float s_red[OAT_NW][32];
    __shared__ int s_qb;
    __shared__ int s_count;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long n_qb = (long long)P.Q * P.NB;

    for (long long item = blockIdx.x; item < P.n_items; item += gridDim.x) {
        if (tid == 0) {                                   // which (q, b) owns this item
            long long lo = 0, hi = n_qb;                  // prefix[lo] <= item < prefix[hi]
            while (hi - lo > 1) {
                const long long mid = (lo + hi) >> 1;
                if (P.item_prefix[mid] <= item) lo = mid; else hi = mid;
            }
            s_qb = (int)lo;
        }
        __syncthreads();
        const int qb = s_qb;
        const int q = qb / P.NB, b = qb - q * P.NB;
        if (tid < 12) {
            const double v = P.frame[(size_t)q * 12 + tid];
            s_frame[tid] = v;
            s_framef[tid] = (float)v;
        }
        const OatBand band = P.band[b];
        const int n_rings_qb = P.qb_rings[qb];
        const OatRing *__restrict__ ring = P.ring + band.ring_ofs;
        const int n_cand = ring[n_rings_qb].cum;          // sentinel-safe: entry n_rings_qb exists
        const long long c_begin = (item - P.item_prefix[qb]) * (long long)OAT_CH;
        const int c_end = (int)min((long long)n_cand, c_begin + OAT_CH);

        const LaneCtx L = lane_setup<MODE>(P, band, q, lane, y);
        float acc = 0.f;
        unsigned cnt = 0;
        __syncthreads();                                  // s_frame ready
        // every warp maps lane -> k the same way, so this vote is uniform over the block:
        // a band whose 32 data values give g' = 0 contributes exactly nothing to H^T y
        const bool live = (MODE != 1) || __any_sync(0xffffffffu, L.coef != 0.f);

        for (int sb = (int)c_begin; live && sb < c_end; sb += OAT_SB) {
            if (tid == 0) s_count = 0;
            __syncthreads();
            // ------------------------------------------------------------ build
            const int sb_end = min(sb + OAT_SB, c_end);
            for (int c = sb + tid; c < sb_end; c += OAT_NT) {
                int lo = 0, hi = n_rings_qb;              // ring r: cum[r] <= c < cum[r+1]
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (ring[mid].cum <= c) lo = mid; else hi = mid;
                }
                const OatRing R = ring[lo];
                const int j = c - R.cum;
                // cheap fp32 pre-test (2.7x more candidates than hits in this schedule)
                float sp, cp;
                sincospif(2.0f * (float)j / (float)R.N, &sp, &cp);
                const float stf = (float)R.st, ctf = (float)R.ct;
                const float lx = stf * cp, ly = stf * sp;
                bool hit = true;
                const float lim[3] = {(float)P.nx + 1.01f, (float)P.ny + 1.01f, (float)P.nz + 1.01f};
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const float ua = lx * s_framef[a] + ly * s_framef[3 + a] + ctf * s_framef[6 + a];
                    const float p0 = fmaf(band.s_lo, ua, s_framef[9 + a]);
                    const float p1 = fmaf(band.s_hi, ua, s_framef[9 + a]);
                    hit = hit && (fmaxf(p0, p1) >= -0.01f) && (fminf(p0, p1) <= lim[a]);
                }
                if (!hit) continue;
                Entry e;
                if (!make_entry(P, band, R, j, s_frame, e)) continue;
                list[atomicAdd(&s_count, 1)] = e;
            }
            __syncthreads();
            // ------------------------------------------------------------ consume
            consume_list<MODE, VAR>(P, list, s_count, warp, lane, L, xpad, xacc, acc, cnt);
            __syncthreads();                              // list is rebuilt next round
        }
        item_epilogue<MODE>(P, q, L, acc, cnt, warp, lane, s_red, g, counter);
        __syncthreads();                                  // s_qb, s_frame, s_red reused by the next item
    }
}

// ------------------------------------------------------------------------------------------------
// Schedule 1: work item = PATCH = (q, band, block of OAT_RI rings, azimuth sector): a compact piece of
// shell, ~32 x 32 x (B c dt / ds) voxels.  Items are generated and culled on the device at geometry
// creation and sorted by the Morton code of their position, so the blocks in flight at any time all
// work inside the same small sub-volume: the volume / the accumulators they touch stay in L1/L2.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void unpack_item(unsigned long long v, int &q, int &b, int &rb, int &s)
{
    s = (int)(v & 0xffffu);
    rb = (int)((v >> 16) & 0x3ffu);
    b = (int)((v >> 26) & 0xfffu);
    q = (int)(v >> 38);
}

template <int MODE, int VAR>
__global__ void __launch_bounds__(OAT_NT, 3)
oat_patch_kernel(const OatDev P, const float *__restrict__ xpad, float *__restrict__ xacc,
                 const float *__restrict__ y, double *__restrict__ g, unsigned long long *__restrict__ counter)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Entry *list = reinterpret_cast<Entry *>(smem_raw);
    __shared__ double s_frame[12];
    __shared__ float s_red[OAT_NW][32];
    __shared__ float s_delta[32], s_coef[32];
    __shared__ int s_count;
    __shared__ int s_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (long long item = blockIdx.x; item < P.n_patches; item += gridDim.x) {
        int q, b, rb, sec;
        unpack_item(P.patches[item], q, b, rb, sec);
        if (tid < 12) s_frame[tid] = P.frame[(size_t)q * 12 + tid];
        if (tid == 0) s_count = 0;
        const OatBand band = P.band[b];
        const OatRing *__restrict__ ring = P.ring + band.ring_ofs;
        const int r0 = rb * OAT_RI;
        const int r1 = min(r0 + OAT_RI, P.qb_rings[(size_t)q * P.NB + b]);
        const int S = P.rb_sectors[band.rb_ofs + rb];
        const LaneCtx L = lane_setup<MODE>(P, band, q, lane, y);
        if (MODE == 1 && VAR == 3 && warp == 0) { s_delta[lane] = L.delta; s_coef[lane] = L.active ? L.coef : 0.f; }
        float acc = 0.f;
        unsigned cnt = 0;
        __syncthreads();
        const bool live = (MODE != 1) || __any_sync(0xffffffffu, L.coef != 0.f);
        if (live) {
            // ---------------------------------------------------------------- build
            for (int t = tid; t < OAT_RI * OAT_RJ; t += OAT_NT) {
                const int r = r0 + t / OAT_RJ, jl = t % OAT_RJ;
                if (r >= r1) break;
                const OatRing R = ring[r];
                const int j0 = (int)(((long long)R.N * sec + S - 1) / S);
                const int j1 = (int)(((long long)R.N * (sec + 1) + S - 1) / S);
                if (j0 + jl >= j1) continue;
                Entry e;
                if (!make_entry(P, band, R, j0 + jl, s_frame, e)) continue;
                list[atomicAdd(&s_count, 1)] = e;
            }
            __syncthreads();
            // ---------------------------------------------------------------- consume
            if (MODE == 1 && VAR == 3) consume_march(P, list, s_count, tid, band.nk, s_delta, s_coef, xacc);
            else consume_list<MODE, ((MODE == 1 && VAR == 3) ? 2 : VAR)>(P, list, s_count, warp, lane, L, xpad, xacc, acc, cnt);
        }
        item_epilogue<MODE>(P, q, L, acc, cnt, warp, lane, s_red, g, counter);
        if (MODE == 0) {
            // Fused step A4 (Eq. 3 L63 / Eq. 13): the block that completes the LAST patch of transducer q
            // turns the finished fp64 row g[q,:] into pressure, y_k = kappa (g_{k+1}/t_{k+1} - g_{k-1}/t_{k-1})/(2 dt).
            // Pattern: every lane fences its own atomics, then one lane counts the patch as done.
            if (warp == 0) {
                __threadfence();
                __syncwarp();
                if (lane == 0) s_last = (atomicAdd(&P.q_done[q], 1) + 1 == P.q_count[q]) ? 1 : 0;
            }
            __syncthreads();
            if (s_last) {
                __threadfence();
                const double *gq = g + (size_t)q * P.K;
                float *yq = xacc + (size_t)q * P.K;          // MODE 0: xacc is the output data vector y
                for (int k = tid; k < P.K; k += OAT_NT) {
                    double sp = 0.0, sm = 0.0;
                    if (k + 1 < P.K) { const double t = P.t0 + (double)(k + 1) * P.dt; if (t > 0.0) sp = __ldcg(gq + k + 1) / t; }
                    if (k - 1 >= 0) { const double t = P.t0 + (double)(k - 1) * P.dt; if (t > 0.0) sm = __ldcg(gq + k - 1) / t; }
                    yq[k] = (float)(P.kappa * (sp - sm) / (2.0 * P.dt));
                }
            }
        }
        __syncthreads();
    }
}

// direction table (once per geometry): one block per (band, ring); see OatDev::dir
__global__ void oat_dir_table_kernel(const OatDev P, double2 *__restrict__ dir)
{
    const OatBand band = P.band[blockIdx.y];
    for (int r = blockIdx.x; r < band.dir_rings; r += gridDim.x) {
        const OatRing R = P.ring[band.ring_ofs + r];
        for (int j = threadIdx.x; j < R.N; j += blockDim.x) {
            double sd, cd;
            sincospi(2.0 * (double)j / (double)R.N, &sd, &cd);        // same expression as make_entry()
            dir[band.dir_ofs + R.cum + j] = make_double2(R.st * cd, R.st * sd);
        }
    }
}

// S7 with the rho^2 of S8 folded in: coef[q,k] = kappa (y[k-1] - y[k+1]) / (2 dt) / t_k * rho_k^2, 0 where t_k <= 0
__global__ void oat_coef_kernel(const OatDev P, const float *__restrict__ y, float *__restrict__ coef)
{
    const long long n = (long long)P.Q * P.K;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int k = (int)(i % P.K);
        const double tk = P.t0 + (double)k * P.dt, rho = P.c * tk;
        const float ym = (k - 1 >= 0) ? y[i - 1] : 0.f;
        const float yp = (k + 1 < P.K) ? y[i + 1] : 0.f;
        const double sp = P.kappa * ((double)ym - (double)yp) / (2.0 * P.dt);   // Eq. 22
        coef[i] = rho > 0.0 ? (float)(sp / tk * rho * rho) : 0.f;
    }
}

// probe for oat_measure_red_rate(): every lane adds a float4 into its own pseudo-random 32-byte sector
__global__ void oat_red_probe_kernel(float4 *__restrict__ buf, unsigned n16, int iters)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        s = s * 1664525u + 1013904223u;
        const unsigned h = (s >> 4) + lane * 2654435761u;
        const unsigned r = ((h ^ (h >> 13)) * 0x9E3779B1u) % (n16 / 2);
        red_add_v4(buf + 2 * (size_t)r, 1.f, 1.f, 1.f, 1.f);
    }
}

// probe for oat_measure_gather_rate(): every lane loads its own pseudo-random 32-byte sector (one 256-bit load, the
// access of consume_march_fwd), four independent loads in flight per thread; the sum keeps the loads alive
__global__ void oat_gather_probe_kernel(const float4 *__restrict__ buf, unsigned n16, int iters, float *__restrict__ sink)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 54321u;
    float acc = 0.f;
    for (int i = 0; i < iters; ++i) {
        float v[4][8];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s = s * 1664525u + 1013904223u;
            const unsigned h = (s >> 4) + lane * 2654435761u;
            const unsigned r = ((h ^ (h >> 13)) * 0x9E3779B1u) % (n16 / 2);
            asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(v[u][0]), "=f"(v[u][1]), "=f"(v[u][2]), "=f"(v[u][3]), "=f"(v[u][4]), "=f"(v[u][5]), "=f"(v[u][6]), "=f"(v[u][7])
                         : "l"(buf + 2 * (size_t)r));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) acc += v[u][0] + v[u][7];
    }
    if (acc == 12345.678f) sink[0] = acc;
}

// probe for oat_measure_gather_rate_ex(): `active` of the 32 lanes load one pseudo-random sector each, ONE load in flight
// per thread (its result is consumed before the next is issued) -- the request shape of the marching loop of H;
// dynamic shared memory (unused) sets the shared-memory carve-out and with it the size of L1
__global__ void __launch_bounds__(128, 8) oat_gather_probe_ex_kernel(const float4 *__restrict__ buf, unsigned nsec, int iters, int active, float *__restrict__ sink)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 54321u;
    float acc = 0.f;
    const bool act = (int)((lane * 7) & 31) < active;
    for (int i = 0; i < iters; ++i) {
        float v[8];
        s = s * 1664525u + 1013904223u;
        const unsigned h = (s >> 4) + lane * 2654435761u;
        const unsigned r = ((h ^ (h >> 13)) * 0x9E3779B1u) & (nsec - 1);      // nsec is a power of two
        if (act) {
            asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                         : "l"(buf + 2 * (size_t)r));
            acc += v[0] + v[7];
        }
    }
    if (acc == 12345.678f) sink[0] = acc;
}

// probe for oat_measure_red_rate_ex(): RED.128 with a chosen address pattern within the warp
__global__ void oat_red_probe_ex_kernel(float4 *__restrict__ buf, unsigned n16, int iters, int pattern)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        s = s * 1664525u + 1013904223u;
        const unsigned wbase = ((s >> 4) ^ (s >> 17)) * 0x9E3779B1u;       // the same for all lanes of the warp
        unsigned r;
        if (pattern == 0) { const unsigned h = (s >> 4) + lane * 2654435761u; r = (h ^ (h >> 13)) * 0x9E3779B1u; }   // every lane its own record
        else if (pattern == 1) r = wbase + lane;                           // 32 consecutive records = 16 sectors in 4 lines
        else if (pattern == 2) r = wbase + lane * 8;                       // one record per 128-byte line, 32 lines
        else if (pattern == 3) r = wbase + (lane >> 1) * 64 + (lane & 1);  // lane pairs share a sector, pairs 1 KB apart
        else r = wbase + (lane >> 3) * 1024 + (lane & 7);                  // 4 scattered lines of 8 records
        red_add_v4(buf + (r % n16), 1.f, 1.f, 1.f, 1.f);
    }
}

// number of patches per transducer (for the fused time-difference epilogue)
__global__ void oat_count_patches_kernel(const unsigned long long *__restrict__ patches, long long n, int *__restrict__ q_count)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        atomicAdd(&q_count[(int)(patches[i] >> 38)], 1);
}

// Patch generation (once per geometry): one block per (q, band); threads stride over (ring block,
// sector); a patch whose bounding sphere can meet the padded node box is appended as
// (Morton key of its centre, packed descriptor).
__device__ __forceinline__ unsigned part1by2(unsigned x)
{
    x &= 0x3ffu;
    x = (x | (x << 16)) & 0x30000ffu;
    x = (x | (x << 8)) & 0x300f00fu;
    x = (x | (x << 4)) & 0x30c30c3u;
    x = (x | (x << 2)) & 0x9249249u;
    return x;
}

__global__ void oat_gen_patches_kernel(const OatDev P, unsigned *__restrict__ keys, unsigned long long *__restrict__ vals,
                                       unsigned long long *__restrict__ n_out, unsigned long long cap, int shift)
{
    const int qb = blockIdx.x;
    const int q = qb / P.NB, b = qb - q * P.NB;
    const int nr = P.qb_rings[qb];
    if (nr <= 0) return;
    const OatBand band = P.band[b];
    const OatRing *__restrict__ ring = P.ring + band.ring_ofs;
    const double *f = P.frame + (size_t)q * 12;
    const int n_rb = (nr + OAT_RI - 1) / OAT_RI;
    // flatten (rb, sector) with a running offset per ring block
    int total = 0;
    for (int rb = 0; rb < n_rb; ++rb) total += P.rb_sectors[band.rb_ofs + rb];
    for (int t = threadIdx.x; t < total; t += blockDim.x) {
        int rb = 0, sec = t;
        while (sec >= P.rb_sectors[band.rb_ofs + rb]) { sec -= P.rb_sectors[band.rb_ofs + rb]; ++rb; }
        const int S = P.rb_sectors[band.rb_ofs + rb];
        const int r0 = rb * OAT_RI, r1 = min(r0 + OAT_RI, nr);
        // patch centre direction and angular radius
        const double th0 = (double)(r0 + 1) * band.dtheta, th1 = (double)r1 * band.dtheta;   // ring index r <-> theta = (r+1) dtheta
        const double thc = 0.5 * (th0 + th1);
        const double phc = 2.0 * 3.14159265358979323846 * ((double)sec + 0.5) / (double)S;
        const double smax = fmax(sin(th0), fmax(sin(th1), (th0 < 1.5707963267948966 && th1 > 1.5707963267948966) ? 1.0 : 0.0));
        const double half_th = 0.5 * (th1 - th0) + band.dtheta;
        const double half_ph = (3.14159265358979323846 / (double)S + 6.3 / (double)ring[r0].N) * smax;
        const double gamma = sqrt(half_th * half_th + half_ph * half_ph);
        double sc, cc; sincos(phc, &sc, &cc);
        const double st = sin(thc), ct = cos(thc);
        double cen[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double ua = st * cc * f[a] + st * sc * f[3 + a] + ct * f[6 + a];
            cen[a] = f[9 + a] + band.s_mid * ua;             // padded voxel coordinates
        }
        const double rad = (double)band.s_hi * fmin(gamma, 3.2) * 1.02 + 0.5 * ((double)band.s_hi - (double)band.s_lo) + 2.0;
        const double hi[3] = {(double)P.nx + 1.0, (double)P.ny + 1.0, (double)P.nz + 1.0};
        double d2 = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double d = cen[a] < 0.0 ? -cen[a] : (cen[a] > hi[a] ? cen[a] - hi[a] : 0.0);
            d2 += d * d;
        }
        if (d2 > rad * rad) continue;
        unsigned cx = (unsigned)fmin(fmax(cen[0], 0.0), hi[0]) >> shift, cy = (unsigned)fmin(fmax(cen[1], 0.0), hi[1]) >> shift,
                 cz = (unsigned)fmin(fmax(cen[2], 0.0), hi[2]) >> shift;
        const unsigned key = part1by2(cx) | (part1by2(cy) << 1) | (part1by2(cz) << 2);
        const unsigned long long slot = atomicAdd(n_out, 1ULL);
        if (slot < cap) {
            keys[slot] = key;
            vals[slot] = ((unsigned long long)q << 38) | ((unsigned long long)b << 26) | ((unsigned long long)rb << 16) | (unsigned long long)sec;
        }
    }
}

// xpad[z+1][y+1][x+1] = x[z][y][x], zero elsewhere (reading G5: zero padding by one node)
__global__ void oat_pad_kernel(const OatDev P, const float *__restrict__ x, float *__restrict__ xpad)
{
    const long long n = (long long)P.pz * P.pxy;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int xx = (int)(i % P.px);
        const long long r = i / P.px;
        const int yy = (int)(r % P.py), zz = (int)(r / P.py);
        float v = 0.f;
        if (xx >= 1 && xx <= P.nx && yy >= 1 && yy <= P.ny && zz >= 1 && zz <= P.nz)
            v = x[((size_t)(zz - 1) * P.ny + (yy - 1)) * P.nx + (xx - 1)];
        xpad[i] = v;
    }
}

// quad arrays from x: array p holds quads with origin (2a + (p&1), 2b + (p>>1)) in padded coordinates
__global__ void oat_pad_quads_kernel(const OatDev P, const float *__restrict__ x, float4 *__restrict__ quads)
{
    const long long n = 4LL * P.pz * P.qplane;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int a = (int)(i % P.qx);
        long long r = i / P.qx;
        const int b = (int)(r % P.qy); r /= P.qy;
        const int z = (int)(r % P.pz);
        const int par = (int)(r / P.pz);
        const int x0 = 2 * a + (par & 1), y0 = 2 * b + (par >> 1);
        float v[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int X = x0 + (c & 1), Y = y0 + (c >> 1);      // padded coordinates; node = (X-1, Y-1, z-1)
            v[c] = (X >= 1 && X <= P.nx && Y >= 1 && Y <= P.ny && z >= 1 && z <= P.nz)
                       ? x[((size_t)(z - 1) * P.ny + (Y - 1)) * P.nx + (X - 1)] : 0.f;
        }
        quads[i] = make_float4(v[0], v[1], v[2], v[3]);
    }
}

// octet arrays from x: array p = (px | py<<1 | pz<<2) holds 2x2x2 bricks with origin (2a+px, 2b+py, 2c+pz)
// in padded coordinates, 8 floats = one aligned 32-byte record = all 8 corners of the cell at that origin
__global__ void oat_pad_octs_kernel(const OatDev P, const float *__restrict__ x, float4 *__restrict__ octs)
{
    const long long n = 8LL * P.oz * P.qplane;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int a = (int)(i % P.qx);
        long long r = i / P.qx;
        const int b = (int)(r % P.qy); r /= P.qy;
        const int c = (int)(r % P.oz);
        const int par = (int)(r / P.oz);
        const int x0 = 2 * a + (par & 1), y0 = 2 * b + ((par >> 1) & 1), z0 = 2 * c + (par >> 2);
        float v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int X = x0 + (k & 1), Y = y0 + ((k >> 1) & 1), Z = z0 + (k >> 2);
            v[k] = (X >= 1 && X <= P.nx && Y >= 1 && Y <= P.ny && Z >= 1 && Z <= P.nz)
                       ? x[((size_t)(Z - 1) * P.ny + (Y - 1)) * P.nx + (X - 1)] : 0.f;
        }
        octs[2 * i] = make_float4(v[0], v[1], v[2], v[3]);
        octs[2 * i + 1] = make_float4(v[4], v[5], v[6], v[7]);
    }
}

// x[n] = sum over the 4 parity arrays of the quad component that is node n (every node is in exactly
// one quad of each array)
__global__ void oat_unquad_kernel(const OatDev P, const float4 *__restrict__ quads, float *__restrict__ x)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int X = (int)(i % P.nx) + 1;
        const long long r = i / P.nx;
        const int Y = (int)(r % P.ny) + 1, Z = (int)(r / P.ny) + 1;
        float sum = 0.f;
#pragma unroll
        for (int par = 0; par < 4; ++par) {
            const int px = par & 1, py = par >> 1;
            const int a = (X - px) >> 1, b = (Y - py) >> 1;
            const int c = (X - px - 2 * a) + 2 * (Y - py - 2 * b);
            const float4 q = quads[((size_t)(par * P.pz + Z) * P.qy + b) * P.qx + a];
            sum += c == 0 ? q.x : c == 1 ? q.y : c == 2 ? q.z : q.w;
        }
        x[i] = sum;
    }
}

// x[n] = sum over the three orientations of the 4 face-quad components that are node n (backproject variant 4):
// every node sits in the quads (ib, ic) in {pb-1, pb} x {pc-1, pc} of plane pa, as component (pb-ib) + 2 (pc-ic)
__global__ void oat_unface_kernel(const OatDev P, const float4 *__restrict__ faces, float *__restrict__ x)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int p[3] = {(int)(i % P.nx) + 1, (int)((i / P.nx) % P.ny) + 1, (int)(i / ((long long)P.nx * P.ny)) + 1};
        float sum = 0.f;
#pragma unroll
        for (int o = 0; o < 3; ++o) {
            const int pa = p[o], pb = p[(o + 1) % 3], pc = p[(o + 2) % 3];
            const float4 *q = faces + P.f_base[o];
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                const int ib = pb - (d & 1), ic = pc - (d >> 1);
                const float4 v = q[((long long)pa * P.f_nc[o] + ic) * P.f_nb[o] + ib];
                sum += d == 0 ? v.x : d == 1 ? v.y : d == 2 ? v.z : v.w;
            }
        }
        x[i] = sum;
    }
}

// same padded volume written into the 2-D slice atlas (slice z at column z & mask, row z >> shift)
__global__ void oat_pad_atlas_kernel(const OatDev P, const float *__restrict__ x, cudaSurfaceObject_t surf)
{
    const long long n = (long long)P.pz * P.pxy;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int xx = (int)(i % P.px);
        const long long r = i / P.px;
        const int yy = (int)(r % P.py), zz = (int)(r / P.py);
        float v = 0.f;
        if (xx >= 1 && xx <= P.nx && yy >= 1 && yy <= P.ny && zz >= 1 && zz <= P.nz)
            v = x[((size_t)(zz - 1) * P.ny + (yy - 1)) * P.nx + (xx - 1)];
        surf2Dwrite(v, surf, (int)sizeof(float) * ((zz & P.atlas_mask) * P.px + xx), (zz >> P.atlas_shift) * P.py + yy);
    }
}

__global__ void oat_unpad_kernel(const OatDev P, const float *__restrict__ xpad, float *__restrict__ x)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int xx = (int)(i % P.nx);
        const long long r = i / P.nx;
        const int yy = (int)(r % P.ny), zz = (int)(r / P.ny);
        x[i] = xpad[((size_t)(zz + 1) * P.py + (yy + 1)) * P.px + (xx + 1)];
    }
}

// S6: y_k = kappa (g_{k+1}/t_{k+1} - g_{k-1}/t_{k-1}) / (2 dt), zero extension, g/t := 0 at t <= 0
__global__ void oat_diff_kernel(const OatDev P, const double *__restrict__ g, float *__restrict__ y)
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

__global__ void oat_dot_kernel(const float *__restrict__ a, const float *__restrict__ b, long long n, double *out)
{
    double s = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        s += (double)a[i] * (double)b[i];
    s = warp_sum(s);
    __shared__ double sh[32];
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
        v = warp_sum(v);
        if (threadIdx.x == 0) atomicAdd(out, v);
    }
}

__global__ void oat_axpy_kernel(float alpha, const float *__restrict__ x, float *__restrict__ y, long long n)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        y[i] = fmaf(alpha, x[i], y[i]);
}

__global__ void oat_xpay_kernel(const float *__restrict__ x, float beta, float *__restrict__ y, long long n)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        y[i] = fmaf(beta, y[i], x[i]);
}

// Row NEXT-1, EIR operator.  ADJ = 0: Eq. (14), out[q,k] = sum_m he[m] in[q, k-1-m]; ADJ = 1: Eq. (21),
// out[q,k] = sum_m he[m] in[q, k+1+m]; he[m] given for m = 0..L-1, `in` zero outside [0, K) (reading G20).
// One block = one transducer row x a tile of OAT_ET outputs; the taps and the input window of the tile sit in
// shared memory; every output is one fixed-order fp32 FMA chain over the taps (deterministic).
#define OAT_ET 256
template <int ADJ>
__global__ void __launch_bounds__(OAT_ET)
oat_eir_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ he, int L, int K)
{
    extern __shared__ float sm[];
    float *s_he = sm, *s_in = sm + L;                      // window: OAT_ET + L samples
    const int q = blockIdx.y, k0 = blockIdx.x * OAT_ET, t = threadIdx.x;
    const float *row = in + (size_t)q * K;
    for (int m = t; m < L; m += OAT_ET) s_he[m] = he[m];
    // ADJ = 0: window sample j <-> k0 - L + j  (inputs k-1-m, m < L, of outputs k0..k0+ET-1: k0-L .. k0+ET-2)
    // ADJ = 1: window sample j <-> k0 + 1 + j  (inputs k+1+m: k0+1 .. k0+ET+L-1)
    const int base = ADJ ? k0 + 1 : k0 - L;
    for (int j = t; j < OAT_ET + L; j += OAT_ET) {
        const int kk = base + j;
        s_in[j] = (kk >= 0 && kk < K) ? row[kk] : 0.f;
    }
    __syncthreads();
    const int k = k0 + t;
    if (k >= K) return;
    float acc = 0.f;
    if (ADJ) { for (int m = 0; m < L; ++m) acc = fmaf(s_he[m], s_in[t + m], acc); }
    else     { for (int m = 0; m < L; ++m) acc = fmaf(s_he[m], s_in[t + L - 1 - m], acc); }
    out[(size_t)q * K + k] = acc;
}

// Row NEXT-1, smoothness penalty (Eq. 34, reading G21): out = beta out + alpha L x with R(x) = x^T L x,
// (L x)_n = sum over the three axes of (x_n - x_before) + (x_n - x_after), each term only if that neighbour exists.
__global__ void oat_penalty_kernel(const OatDev P, const float *__restrict__ x, float *__restrict__ out, float alpha, float beta)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    const long long sy = P.nx, sz = (long long)P.nx * P.ny;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(i % P.nx);
        const long long r = i / P.nx;
        const int iy = (int)(r % P.ny), iz = (int)(r / P.ny);
        const float c = x[i];
        float s = 0.f;
        if (ix > 0) s += c - x[i - 1];
        if (ix + 1 < P.nx) s += c - x[i + 1];
        if (iy > 0) s += c - x[i - sy];
        if (iy + 1 < P.ny) s += c - x[i + sy];
        if (iz > 0) s += c - x[i - sz];
        if (iz + 1 < P.nz) s += c - x[i + sz];
        out[i] = beta == 0.f ? alpha * s : fmaf(beta, out[i], alpha * s);
    }
}

// Row NEXT-2, filtered backprojection (Eq. 27 L221 with one weight per transducer, readings G23-G25): voxel driven,
// one thread per node of an 8 x 8 x 4 tile, transducers staged through shared memory 256 at a time.  The sample index
// k = floor(k~), k~ = |r_q - r_n| / (c dt) - t_min/dt, is an integer decision and is taken in fp64 like the oracle's
// (the discretisation is discontinuous across integer k~: an fp32 distance, 1e-4 samples off at k~ ~ 2000, would move
// ~1e-4 of all pairs into the neighbouring interval); the two brackets, the interpolation and the sum are fp32, with
// an fp64 total over the chunks of 256 transducers.
#define OAT_FQ 256
__global__ void __launch_bounds__(256)
oat_fbp_kernel(const OatDev P, const float *__restrict__ p, const float *__restrict__ wq, float *__restrict__ x)
{
    __shared__ double s_t[OAT_FQ][3];
    __shared__ float s_w[OAT_FQ];
    const int tid = threadIdx.x;
    const int ix = blockIdx.x * 8 + (tid & 7), iy = blockIdx.y * 8 + ((tid >> 3) & 7), iz = blockIdx.z * 4 + (tid >> 6);
    const bool inside = ix < P.nx && iy < P.ny && iz < P.nz;
    const double vx = (double)ix, vy = (double)iy, vz = (double)iz;   // node coordinates; transducers in the same units
    const double inv_step = 1.0 / P.step, tau = P.t0 / P.dt;
    const float tauf = (float)tau;
    double total = 0.0;
    for (int q0 = 0; q0 < P.Q; q0 += OAT_FQ) {
        const int nq = min(OAT_FQ, P.Q - q0);
        __syncthreads();
        if (tid < nq) {
            const double *f = P.frame + (size_t)(q0 + tid) * 12;
            s_t[tid][0] = f[9] - 1.0; s_t[tid][1] = f[10] - 1.0; s_t[tid][2] = f[11] - 1.0;   // frames hold padded coordinates
            s_w[tid] = wq[q0 + tid];
        }
        __syncthreads();
        if (!inside) continue;
        float acc = 0.f;
#pragma unroll 2
        for (int j = 0; j < nq; ++j) {
            const double dx = vx - s_t[j][0], dy = vy - s_t[j][1], dz = vz - s_t[j][2];
            const double d = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
            const double den = d * inv_step;               // k~ + tau = |r_q - r_n| / (c dt)
            const double kt = den - tau;
            const double kf = floor(kt);
            const int k = (int)kf;
            const bool ok = ((unsigned)k < (unsigned)(P.K - 1)) && den > 0.0;     // k >= 0, k+1 <= K-1 (reading G25)
            const float ktau = (float)kf + tauf;           // k + tau
            const float rden = __fdividef(1.f, (float)den);
            const float a1 = fmaf(-ktau, rden, 1.5f), a0 = fmaf(ktau + 1.f, rden, -1.5f);
            const float *row = p + (size_t)(q0 + j) * P.K;
            const float p0 = ok ? __ldg(row + k) : 0.f, p1 = ok ? __ldg(row + k + 1) : 0.f;
            acc = fmaf(s_w[j], fmaf(a1, p1, a0 * p0), acc);
        }
        total += (double)acc;
    }
    if (inside) x[((size_t)iz * P.ny + iy) * P.nx + ix] = (float)total;
}

// Row NEXT-3, spherical-voxel model in the temporal frequency domain, point-like transducers (Eq. 17-19,
// Eq. 24, Alg. 9; readings G27-G29).  u[q,l] = p0[l] sum_n x_n exp(-j 2 pi f_l d/c) / (2 pi d).
// The phase 2 pi f d / c reaches ~10^3 cycles, so the distance and the phase reduction (frac of f d / c) are fp64; the
// phasor of the first frequency of a group of OAT_SG and the phasor step exp(-j 2 pi df d/c) come from sincospif, the
// other frequencies of the group by complex recurrence (OAT_SG - 1 fp32 rotations, error ~ OAT_SG eps).
#define OAT_SG 16          // frequencies per thread (forward) / per re-seeded group (adjoint)
#define OAT_SV 2048        // voxels per block chunk (forward)
struct OatSph { int nf, n_lg; double f0, df, ds_over_c, ds; };   // ds_over_c: microseconds per node unit of distance

__global__ void __launch_bounds__(128)
oat_sph_fwd_kernel(const OatDev P, const OatSph S, const float *__restrict__ x, const float2 *__restrict__ p0, float *__restrict__ u)
{
    __shared__ float s_x[OAT_SV];
    const long long n_vox = (long long)P.nx * P.ny * P.nz;
    const long long v0 = (long long)blockIdx.y * OAT_SV;
    const int nv = (int)min((long long)OAT_SV, n_vox - v0);
    int any = 0;
    for (int i = threadIdx.x; i < nv; i += blockDim.x) { const float v = x[v0 + i]; s_x[i] = v; any |= (v != 0.f); }
    if (!__syncthreads_or(any)) return;                    // an all-zero chunk contributes nothing
    const long long wi = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (wi >= (long long)P.Q * S.n_lg) return;
    const int q = (int)(wi / S.n_lg), lg = (int)(wi % S.n_lg);
    const int l0 = lg * OAT_SG;
    const double *f = P.frame + (size_t)q * 12;
    const double tx = f[9] - 1.0, ty = f[10] - 1.0, tz = f[11] - 1.0;       // node coordinates (frames hold padded ones)
    const double fa = S.f0 + (double)l0 * S.df;
    float ar[OAT_SG], ai[OAT_SG];
#pragma unroll
    for (int j = 0; j < OAT_SG; ++j) ar[j] = ai[j] = 0.f;
    int ix = (int)(v0 % P.nx), iy = (int)((v0 / P.nx) % P.ny), iz = (int)(v0 / ((long long)P.nx * P.ny));
    for (int i = 0; i < nv; ++i) {
        const float xv = s_x[i];                           // same address for the whole block: a broadcast
        if (xv != 0.f) {                                   // block-uniform branch
            const double dx = (double)ix - tx, dy = (double)iy - ty, dz = (double)iz - tz;
            const double d = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
            if (d > 0.0) {
                const double td = d * S.ds_over_c;         // |r_q - r_n| / c
                const double pa = fa * td, pd = S.df * td; // cycles
                float sr, cr, sz, cz;
                sincospif((float)(-2.0 * (pa - rint(pa))), &sr, &cr);
                sincospif((float)(-2.0 * (pd - rint(pd))), &sz, &cz);
                const float amp = xv / (float)(6.283185307179586 * d * S.ds);
                float er = amp * cr, ei = amp * sr;
#pragma unroll
                for (int j = 0; j < OAT_SG; ++j) {
                    ar[j] += er; ai[j] += ei;
                    const float nr = fmaf(er, cz, -ei * sz);
                    ei = fmaf(er, sz, ei * cz);
                    er = nr;
                }
            }
        }
        if (++ix == P.nx) { ix = 0; if (++iy == P.ny) { iy = 0; ++iz; } }
    }
#pragma unroll
    for (int j = 0; j < OAT_SG; ++j) {
        const int l = l0 + j;
        if (l < S.nf) {
            const float2 c = p0[l];
            float *o = u + 2 * ((size_t)q * S.nf + l);
            atomicAdd(o, ar[j] * c.x - ai[j] * c.y);
            atomicAdd(o + 1, ar[j] * c.y + ai[j] * c.x);
        }
    }
}

// v[q,l] = u[q,l] conj(p0[l])   (the data-side factor of Eq. 24)
__global__ void oat_sph_prep_kernel(const OatSph S, int Q, const float2 *__restrict__ u, const float2 *__restrict__ p0, float2 *__restrict__ v)
{
    const long long n = (long long)Q * S.nf;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float2 a = u[i], c = p0[i % S.nf];
        v[i] = make_float2(a.x * c.x + a.y * c.y, a.y * c.x - a.x * c.y);
    }
}

// x[n] = Re sum_q sum_l v[q,l] exp(+j 2 pi f_l d/c) / (2 pi d)   (Eq. 24, reading G29); one thread per voxel, the rows
// v[q,:] of OAT_SQ transducers staged in shared memory at a time (every thread reads the same element: broadcast)
#define OAT_SQ 4
#define OAT_SL 512         // frequencies per staged slab
__global__ void __launch_bounds__(128)
oat_sph_bwd_kernel(const OatDev P, const OatSph S, const float2 *__restrict__ v, float *__restrict__ x)
{
    __shared__ float2 s_v[OAT_SQ][OAT_SL];
    __shared__ double s_t[OAT_SQ][3];
    const long long n_vox = (long long)P.nx * P.ny * P.nz;
    const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool inside = n < n_vox;
    const int ix = (int)(n % P.nx), iy = (int)((n / P.nx) % P.ny), iz = (int)(n / ((long long)P.nx * P.ny));
    double total = 0.0;
    for (int q0 = 0; q0 < P.Q; q0 += OAT_SQ) {
        const int nq = min(OAT_SQ, P.Q - q0);
        for (int lb = 0; lb < S.nf; lb += OAT_SL) {
            const int nl = min(OAT_SL, S.nf - lb);
            __syncthreads();
            for (int t = threadIdx.x; t < nq * nl; t += blockDim.x) s_v[t / nl][t % nl] = v[(size_t)(q0 + t / nl) * S.nf + lb + t % nl];
            if (threadIdx.x < nq * 3) s_t[threadIdx.x / 3][threadIdx.x % 3] = P.frame[(size_t)(q0 + threadIdx.x / 3) * 12 + 9 + threadIdx.x % 3] - 1.0;
            __syncthreads();
            if (!inside) continue;
            for (int j = 0; j < nq; ++j) {
                const double dx = (double)ix - s_t[j][0], dy = (double)iy - s_t[j][1], dz = (double)iz - s_t[j][2];
                const double d = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
                if (!(d > 0.0)) continue;
                const double td = d * S.ds_over_c, pd = S.df * td;
                float sz, cz;
                sincospif((float)(2.0 * (pd - rint(pd))), &sz, &cz);
                const float amp = 1.f / (float)(6.283185307179586 * d * S.ds);
                float acc = 0.f;
                for (int g0 = 0; g0 < nl; g0 += OAT_SG) {
                    const double pa = (S.f0 + (double)(lb + g0) * S.df) * td;
                    float sr, cr;
                    sincospif((float)(2.0 * (pa - rint(pa))), &sr, &cr);
                    float er = amp * cr, ei = amp * sr;
                    const int ng = min(OAT_SG, nl - g0);
                    if (ng == OAT_SG) {                    // full group: unrolled
#pragma unroll
                        for (int k = 0; k < OAT_SG; ++k) {
                            const float2 vv = s_v[j][g0 + k];
                            acc = fmaf(vv.x, er, fmaf(-vv.y, ei, acc));    // Re(v e)
                            const float nr = fmaf(er, cz, -ei * sz);
                            ei = fmaf(er, sz, ei * cz);
                            er = nr;
                        }
                    } else {
                        for (int k = 0; k < ng; ++k) {
                            const float2 vv = s_v[j][g0 + k];
                            acc = fmaf(vv.x, er, fmaf(-vv.y, ei, acc));
                            const float nr = fmaf(er, cz, -ei * sz);
                            ei = fmaf(er, sz, ei * cz);
                            er = nr;
                        }
                    }
                }
                total += (double)acc;
            }
        }
    }
    if (inside) x[n] = (float)total;
}

inline int grid_for(long long n, int block)
{
    long long g = (n + block - 1) / block;
    const long long cap = 148LL * 16;                     // grid-stride: a few waves over the 148 SMs
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

}  // namespace

void oat_launch_pad(const OatDev &P, const float *x, float *xpad, cudaStream_t st)
{
    const long long n = (long long)P.pz * P.pxy;
    oat_pad_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, x, xpad);
}

void oat_launch_pad_quads(const OatDev &P, const float *x, float4 *quads, cudaStream_t st)
{
    const long long n = 4LL * P.pz * P.qplane;
    oat_pad_quads_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, x, quads);
}

void oat_launch_pad_octs(const OatDev &P, const float *x, float4 *octs, cudaStream_t st)
{
    const long long n = 8LL * P.oz * P.qplane;
    oat_pad_octs_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, x, octs);
}

void oat_launch_unface(const OatDev &P, const float4 *faces, float *x, cudaStream_t st)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    oat_unface_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, faces, x);
}

void oat_launch_unquad(const OatDev &P, const float4 *quads, float *x, cudaStream_t st)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    oat_unquad_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, quads, x);
}

void oat_launch_pad_atlas(const OatDev &P, const float *x, cudaSurfaceObject_t surf, cudaStream_t st)
{
    const long long n = (long long)P.pz * P.pxy;
    oat_pad_atlas_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, x, surf);
}

void oat_launch_unpad(const OatDev &P, const float *xpad, float *x, cudaStream_t st)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    oat_unpad_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, xpad, x);
}

template <int MODE, int VAR>
static cudaError_t launch_ray_t(const OatDev &P, const float *xpad, float *xacc, const float *y, double *g,
                                unsigned long long *counter, cudaStream_t st)
{
    const size_t smem = sizeof(Entry) * OAT_SB;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(oat_ray_kernel<MODE, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e) return e;
        attr_set = true;
    }
    const long long cap = 0x7fffffffLL;
    const unsigned grid = (unsigned)(P.n_items < cap ? P.n_items : cap);
    oat_ray_kernel<MODE, VAR><<<grid, OAT_NT, smem, st>>>(P, xpad, xacc, y, g, counter);
    return cudaGetLastError();
}

template <int MODE, int VAR>
static cudaError_t launch_patch_t(const OatDev &P, const float *xpad, float *xacc, const float *y, double *g,
                                  unsigned long long *counter, cudaStream_t st)
{
    const size_t smem = sizeof(Entry) * OAT_RI * OAT_RJ;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(oat_patch_kernel<MODE, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e) return e;
        attr_set = true;
    }
    const long long cap = 0x7fffffffLL;
    const unsigned grid = (unsigned)(P.n_patches < cap ? P.n_patches : cap);
    oat_patch_kernel<MODE, VAR><<<grid, OAT_NT, smem, st>>>(P, xpad, xacc, y, g, counter);
    return cudaGetLastError();
}

void oat_launch_dir_table(const OatDev &P, int n_bands, double2 *dir, cudaStream_t st)
{
    if (n_bands > 0) oat_dir_table_kernel<<<dim3(256, (unsigned)n_bands), 128, 0, st>>>(P, dir);
}

void oat_launch_red_probe(float4 *buf, unsigned n16, int iters, int blocks, cudaStream_t st)
{
    oat_red_probe_kernel<<<blocks, 256, 0, st>>>(buf, n16, iters);
}

void oat_launch_gather_probe(const float4 *buf, unsigned n16, int iters, int blocks, float *sink, cudaStream_t st)
{
    oat_gather_probe_kernel<<<blocks, 256, 0, st>>>(buf, n16, iters, sink);
}

cudaError_t oat_launch_gather_probe_ex(const float4 *buf, unsigned nsec, int iters, int active, int smem_bytes, int blocks, float *sink, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(oat_gather_probe_ex_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e != cudaSuccess) return e;
    oat_gather_probe_ex_kernel<<<blocks, 128, smem_bytes, st>>>(buf, nsec, iters, active, sink);
    return cudaGetLastError();
}

void oat_launch_red_probe_ex(float4 *buf, unsigned n16, int iters, int pattern, int blocks, cudaStream_t st)
{
    oat_red_probe_ex_kernel<<<blocks, 256, 0, st>>>(buf, n16, iters, pattern);
}

void oat_launch_coef(const OatDev &P, const float *y, float *coef, cudaStream_t st)
{
    const long long n = (long long)P.Q * P.K;
    if (n > 0) oat_coef_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, y, coef);
}

cudaError_t oat_launch_patch(int mode, int variant, const OatDev &P, const float *xpad, float *xacc, const float *y,
                             double *g, unsigned long long *counter, cudaStream_t st)
{
    if (P.n_patches <= 0) return cudaSuccess;
    if (mode == 0) return variant == 3 ? launch_patch_t<0, 3>(P, xpad, xacc, y, g, counter, st)
                        : variant == 2 ? launch_patch_t<0, 2>(P, xpad, xacc, y, g, counter, st)
                        : variant == 1 ? launch_patch_t<0, 1>(P, xpad, xacc, y, g, counter, st)
                                       : launch_patch_t<0, 0>(P, xpad, xacc, y, g, counter, st);
    if (mode == 1) return variant == 3 ? launch_patch_t<1, 3>(P, xpad, xacc, y, g, counter, st)
                        : variant == 2 ? launch_patch_t<1, 2>(P, xpad, xacc, y, g, counter, st)
                        : variant == 1 ? launch_patch_t<1, 1>(P, xpad, xacc, y, g, counter, st)
                                       : launch_patch_t<1, 0>(P, xpad, xacc, y, g, counter, st);
    return launch_patch_t<2, 0>(P, xpad, xacc, y, g, counter, st);
}

// Generates the patch list of a geometry on the device and sorts it by Morton key.  `cap` is the
// host-computed upper bound on the number of patches.  On return *n_patches is the number generated;
// *patches_out is a device buffer the caller owns.
cudaError_t oat_build_patches(const OatDev &P, unsigned long long cap, int shift, int *q_count, unsigned long long **patches_out, long long *n_patches)
{
    *patches_out = nullptr; *n_patches = 0;
    if (cap == 0 || P.Q == 0) return cudaSuccess;
    unsigned *keys = nullptr, *keys2 = nullptr;
    unsigned long long *vals = nullptr, *vals2 = nullptr, *cnt = nullptr;
    void *tmp = nullptr;
    cudaError_t e = cudaSuccess;
    auto cleanup = [&]() { cudaFree(keys); cudaFree(keys2); cudaFree(vals); cudaFree(cnt); cudaFree(tmp); };
#define OAT_TRY(x) do { e = (x); if (e != cudaSuccess) { cleanup(); cudaFree(vals2); return e; } } while (0)
    OAT_TRY(cudaMalloc((void **)&keys, sizeof(unsigned) * cap));
    OAT_TRY(cudaMalloc((void **)&vals, sizeof(unsigned long long) * cap));
    OAT_TRY(cudaMalloc((void **)&cnt, sizeof(unsigned long long)));
    OAT_TRY(cudaMemset(cnt, 0, sizeof(unsigned long long)));
    oat_gen_patches_kernel<<<(unsigned)((long long)P.Q * P.NB), 128>>>(P, keys, vals, cnt, cap, shift);
    OAT_TRY(cudaGetLastError());
    unsigned long long n = 0;
    OAT_TRY(cudaMemcpy(&n, cnt, sizeof(n), cudaMemcpyDeviceToHost));
    if (n > cap) { cleanup(); return cudaErrorInvalidValue; }
    if (n == 0) { cleanup(); return cudaSuccess; }
    OAT_TRY(cudaMalloc((void **)&keys2, sizeof(unsigned) * n));
    OAT_TRY(cudaMalloc((void **)&vals2, sizeof(unsigned long long) * n));
    size_t tmp_bytes = 0;
    OAT_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, vals, vals2, (long long)n, 0, 30));
    OAT_TRY(cudaMalloc(&tmp, tmp_bytes));
    OAT_TRY(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys2, vals, vals2, (long long)n, 0, 30));
    OAT_TRY(cudaDeviceSynchronize());
#undef OAT_TRY
    cleanup();
    if (q_count) {
        oat_count_patches_kernel<<<grid_for((long long)n, 256), 256>>>(vals2, (long long)n, q_count);
        if ((e = cudaDeviceSynchronize()) != cudaSuccess) { cudaFree(vals2); return e; }
    }
    *patches_out = vals2;
    *n_patches = (long long)n;
    return cudaSuccess;
}

cudaError_t oat_launch_ray(int mode, int variant, const OatDev &P, const float *xpad, float *xacc, const float *y,
                           double *g, unsigned long long *counter, cudaStream_t st)
{
    if (P.n_items <= 0) return cudaSuccess;
    if (mode == 0) return variant == 3 ? launch_ray_t<0, 3>(P, xpad, xacc, y, g, counter, st)
                        : variant == 2 ? launch_ray_t<0, 2>(P, xpad, xacc, y, g, counter, st)
                        : variant == 1 ? launch_ray_t<0, 1>(P, xpad, xacc, y, g, counter, st)
                                       : launch_ray_t<0, 0>(P, xpad, xacc, y, g, counter, st);
    if (mode == 1) return variant >= 2 ? launch_ray_t<1, 2>(P, xpad, xacc, y, g, counter, st)
                        : variant == 1 ? launch_ray_t<1, 1>(P, xpad, xacc, y, g, counter, st)
                                       : launch_ray_t<1, 0>(P, xpad, xacc, y, g, counter, st);
    return launch_ray_t<2, 0>(P, xpad, xacc, y, g, counter, st);
}

void oat_launch_diff(const OatDev &P, const double *g, float *y, cudaStream_t st)
{
    const long long n = (long long)P.Q * P.K;
    if (n > 0) oat_diff_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, g, y);
}

cudaError_t oat_launch_eir(int adjoint, const float *in, float *out, const float *he, int L, int Q, int K, cudaStream_t st)
{
    if (Q <= 0 || K <= 0) return cudaSuccess;
    const size_t smem = sizeof(float) * (size_t)(OAT_ET + 2 * L);
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(oat_eir_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(oat_eir_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const dim3 grid((unsigned)((K + OAT_ET - 1) / OAT_ET), (unsigned)Q);
    if (adjoint) oat_eir_kernel<1><<<grid, OAT_ET, smem, st>>>(in, out, he, L, K);
    else oat_eir_kernel<0><<<grid, OAT_ET, smem, st>>>(in, out, he, L, K);
    return cudaGetLastError();
}

void oat_launch_fbp(const OatDev &P, const float *p, const float *wq, float *x, cudaStream_t st)
{
    const dim3 grid((unsigned)((P.nx + 7) / 8), (unsigned)((P.ny + 7) / 8), (unsigned)((P.nz + 3) / 4));
    oat_fbp_kernel<<<grid, 256, 0, st>>>(P, p, wq, x);
}

void oat_launch_sph_fwd(const OatDev &P, int nf, double f0, double df, double ds, double c, const float *x, const float2 *p0, float *u, cudaStream_t st)
{
    OatSph S; S.nf = nf; S.n_lg = (nf + OAT_SG - 1) / OAT_SG; S.f0 = f0; S.df = df; S.ds = ds; S.ds_over_c = ds / c;
    const long long n_vox = (long long)P.nx * P.ny * P.nz, work = (long long)P.Q * S.n_lg;
    if (n_vox <= 0 || work <= 0) return;
    const dim3 grid((unsigned)((work + 127) / 128), (unsigned)((n_vox + OAT_SV - 1) / OAT_SV));
    oat_sph_fwd_kernel<<<grid, 128, 0, st>>>(P, S, x, p0, u);
}

void oat_launch_sph_bwd(const OatDev &P, int nf, double f0, double df, double ds, double c, const float2 *u, const float2 *p0, float2 *v, float *x, cudaStream_t st)
{
    OatSph S; S.nf = nf; S.n_lg = (nf + OAT_SG - 1) / OAT_SG; S.f0 = f0; S.df = df; S.ds = ds; S.ds_over_c = ds / c;
    const long long n_vox = (long long)P.nx * P.ny * P.nz, n = (long long)P.Q * nf;
    if (n > 0) oat_sph_prep_kernel<<<grid_for(n, 256), 256, 0, st>>>(S, P.Q, u, p0, v);
    if (n_vox > 0) oat_sph_bwd_kernel<<<(unsigned)((n_vox + 127) / 128), 128, 0, st>>>(P, S, v, x);
}

void oat_launch_penalty(const OatDev &P, const float *x, float *out, float alpha, float beta, cudaStream_t st)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    if (n > 0) oat_penalty_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, x, out, alpha, beta);
}

void oat_launch_dot(const float *a, const float *b, long long n, double *out, cudaStream_t st)
{
    if (n > 0) oat_dot_kernel<<<grid_for(n, 256), 256, 0, st>>>(a, b, n, out);
}

void oat_launch_axpy(float alpha, const float *x, float *y, long long n, cudaStream_t st)
{
    if (n > 0) oat_axpy_kernel<<<grid_for(n, 256), 256, 0, st>>>(alpha, x, y, n);
}

void oat_launch_xpay(const float *x, float beta, float *y, long long n, cudaStream_t st)
{
    if (n > 0) oat_xpay_kernel<<<grid_for(n, 256), 256, 0, st>>>(x, beta, y, n);
}
