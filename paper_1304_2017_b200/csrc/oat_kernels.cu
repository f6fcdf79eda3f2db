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

namespace {

struct __align__(16) Entry {
    float4 a;   // anchor fraction (x,y,z) in [-0.5,0.5], omega
    float4 u;   // direction (x,y,z) in voxel axes, unused
    int4 i;     // anchor integer node offset in the padded volume (x,y,z), unused
};

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

__device__ __forceinline__ bool lane_sample(const OatDev &P, const Entry &e, float delta, Sample &s)
{
    const float tx = fmaf(delta, e.u.x, e.a.x);
    const float ty = fmaf(delta, e.u.y, e.a.y);
    const float tz = fmaf(delta, e.u.z, e.a.z);
    const float flx = floorf(tx), fly = floorf(ty), flz = floorf(tz);
    s.ix = (int)flx + e.i.x;
    s.iy = (int)fly + e.i.y;
    s.iz = (int)flz + e.i.z;
    s.fx = tx - flx;
    s.fy = ty - fly;
    s.fz = tz - flz;
    // padded cell n' in [0, N] <=> xi in [-1, N): the sample touches at least one existing node (S4)
    return ((unsigned)s.ix <= (unsigned)P.nx) & ((unsigned)s.iy <= (unsigned)P.ny) & ((unsigned)s.iz <= (unsigned)P.nz);
}

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

        // lane = time sample of the band
        const int k = band.k0 + lane;
        const double tk = P.t0 + (double)k * P.dt;
        const double rho = P.c * tk;
        const bool active = (lane < band.nk) && (rho > 0.0);
        const float delta = (float)(((double)lane - 0.5 * (double)(P.B - 1)) * P.step);
        float coef = 0.f;                                 // MODE 1: g'_k * rho_k^2  (S7, S8)
        if (MODE == 1 && active) {
            const float ym = (k - 1 >= 0) ? y[(size_t)q * P.K + k - 1] : 0.f;
            const float yp = (k + 1 < P.K) ? y[(size_t)q * P.K + k + 1] : 0.f;
            const double sp = P.kappa * ((double)ym - (double)yp) / (2.0 * P.dt);   // Eq. 22
            coef = (float)(sp / tk * rho * rho);
        }
        float acc = 0.f;
        unsigned cnt = 0;
        __syncthreads();                                  // s_frame ready
        // every warp maps lane -> k the same way, so this vote is uniform over the block:
        // a band whose 32 data values give g' = 0 contributes exactly nothing to H^T y
        const bool live = (MODE != 1) || __any_sync(0xffffffffu, coef != 0.f);

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
                // fp32 pre-test: bounding box of the ray segment against the padded box
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
                // survivors: direction (S3) and anchor in fp64
                double sd, cd;
                sincospi(2.0 * (double)j / (double)R.N, &sd, &cd);
                const double dlx = R.st * cd, dly = R.st * sd, dlz = R.ct;
                Entry e;
                float uu[3], af[3];
                int ai[3];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const double ua = dlx * s_frame[a] + dly * s_frame[3 + a] + dlz * s_frame[6 + a];
                    const double an = s_frame[9 + a] + band.s_mid * ua;
                    const double ar = rint(an);
                    uu[a] = (float)ua;
                    af[a] = (float)(an - ar);
                    ai[a] = (int)ar;
                }
                e.a = make_float4(af[0], af[1], af[2], R.omega);
                e.u = make_float4(uu[0], uu[1], uu[2], 0.f);
                e.i = make_int4(ai[0], ai[1], ai[2], 0);
                const int slot = atomicAdd(&s_count, 1);
                list[slot] = e;
            }
            __syncthreads();
            // ------------------------------------------------------------ consume
            const int n_list = s_count;
            for (int ei = warp; ei < n_list; ei += OAT_NW) {
                const Entry e = list[ei];
                Sample s;
                const bool in = lane_sample(P, e, delta, s) && active;
                if (MODE == 2) { cnt += in ? 1u : 0u; continue; }
                if (MODE == 0) {
                    if (!in) continue;
                    float v000, v100, v010, v110, v001, v101, v011, v111;
                    if (VAR == 0) {                       // 8 scalar loads from the padded linear volume
                        const float *p = xpad + ((size_t)s.iz * P.py + s.iy) * P.px + s.ix;
                        v000 = __ldg(p); v100 = __ldg(p + 1);
                        v010 = __ldg(p + P.px); v110 = __ldg(p + P.px + 1);
                        const float *p1 = p + P.pxy;
                        v001 = __ldg(p1); v101 = __ldg(p1 + 1);
                        v011 = __ldg(p1 + P.px); v111 = __ldg(p1 + P.px + 1);
                    } else {                              // 2 texture gathers (tld4) from the slice atlas
                        const int z1 = s.iz + 1;
                        const float tx = (float)s.ix + 1.0f, ty = (float)s.iy + 1.0f;   // between texel centres: exact 2x2 footprint
                        const float ax0 = (float)((s.iz & P.atlas_mask) * P.px), ay0 = (float)((s.iz >> P.atlas_shift) * P.py);
                        const float ax1 = (float)((z1 & P.atlas_mask) * P.px), ay1 = (float)((z1 >> P.atlas_shift) * P.py);
                        const float4 lo = tex2Dgather<float4>(P.tex, tx + ax0, ty + ay0, 0);
                        const float4 hi = tex2Dgather<float4>(P.tex, tx + ax1, ty + ay1, 0);
                        // gather order: x = (i, j+1), y = (i+1, j+1), z = (i+1, j), w = (i, j)
                        v000 = lo.w; v100 = lo.z; v010 = lo.x; v110 = lo.y;
                        v001 = hi.w; v101 = hi.z; v011 = hi.x; v111 = hi.y;
                    }
                    const float a00 = fmaf(s.fx, v100 - v000, v000);
                    const float a10 = fmaf(s.fx, v110 - v010, v010);
                    const float a01 = fmaf(s.fx, v101 - v001, v001);
                    const float a11 = fmaf(s.fx, v111 - v011, v011);
                    const float b0 = fmaf(s.fy, a10 - a00, a00);
                    const float b1 = fmaf(s.fy, a11 - a01, a01);
                    acc = fmaf(e.a.w, fmaf(s.fz, b1 - b0, b0), acc);
                } else if (MODE == 1) {
                    if (VAR == 0) { if (!in) continue; }
                    else if (!__any_sync(0xffffffffu, in)) continue;
                    const size_t idx = ((size_t)s.iz * P.py + s.iy) * P.px + s.ix;
                    const float cw = in ? coef * e.a.w : 0.f;
                    const float wz1 = s.fz * cw, wz0 = cw - wz1;
                    const float gx = 1.f - s.fx, gy = 1.f - s.fy;
                    float w[8] = {gx * gy * wz0, s.fx * gy * wz0, gx * s.fy * wz0, s.fx * s.fy * wz0,
                                  gx * gy * wz1, s.fx * gy * wz1, gx * s.fy * wz1, s.fx * s.fy * wz1};
                    bool writer = in;
                    if (VAR == 1) {
                        // Lanes step along one ray, so lanes that fall into the same cell are CONSECUTIVE:
                        // sum each run into its first lane (segmented suffix sum by shuffles) and let only
                        // run heads issue the 8 atomics (~3x fewer L2 atomic operations).
                        const unsigned cell = in ? (unsigned)idx : (0xfffffff0u - (unsigned)lane);
                        const unsigned prev = __shfl_up_sync(0xffffffffu, cell, 1);
                        const bool head = (lane == 0) || (cell != prev);
                        const unsigned heads = __ballot_sync(0xffffffffu, head);
                        const unsigned above = (lane == 31) ? 0u : (heads & ~((2u << lane) - 1u));
                        const int run_end = above ? (__ffs(above) - 2) : 31;
                        const unsigned maxrun = __reduce_max_sync(0xffffffffu, head ? (unsigned)(run_end - lane + 1) : 0u);
                        for (unsigned d = 1; d < maxrun; d <<= 1) {
                            const bool take = (lane + (int)d) <= run_end;
#pragma unroll
                            for (int c = 0; c < 8; ++c) {
                                const float o = __shfl_down_sync(0xffffffffu, w[c], d);
                                if (take) w[c] += o;
                            }
                        }
                        writer = in && head;
                    }
                    if (writer) {
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
            __syncthreads();                              // list is rebuilt next round
        }

        // ---------------------------------------------------------------- epilogue
        if (MODE == 0) {
            s_red[warp][lane] = acc;
            __syncthreads();
            if (warp == 0) {
                double sum = 0.0;
#pragma unroll
                for (int w = 0; w < OAT_NW; ++w) sum += (double)s_red[w][lane];
                if (active && sum != 0.0) atomicAdd(&g[(size_t)q * P.K + k], rho * rho * sum);   // S5
            }
        } else if (MODE == 2) {
            const double tot = warp_sum((double)cnt);
            if (lane == 0 && tot > 0) atomicAdd(counter, (unsigned long long)tot);
        }
        __syncthreads();                                  // s_qb, s_frame, s_red reused by the next item
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

cudaError_t oat_launch_ray(int mode, int variant, const OatDev &P, const float *xpad, float *xacc, const float *y,
                           double *g, unsigned long long *counter, cudaStream_t st)
{
    if (P.n_items <= 0) return cudaSuccess;
    if (mode == 0) return variant == 1 ? launch_ray_t<0, 1>(P, xpad, xacc, y, g, counter, st)
                                       : launch_ray_t<0, 0>(P, xpad, xacc, y, g, counter, st);
    if (mode == 1) return variant == 0 ? launch_ray_t<1, 0>(P, xpad, xacc, y, g, counter, st)
                                       : launch_ray_t<1, 1>(P, xpad, xacc, y, g, counter, st);
    return launch_ray_t<2, 0>(P, xpad, xacc, y, g, counter, st);
}

void oat_launch_diff(const OatDev &P, const double *g, float *y, cudaStream_t st)
{
    const long long n = (long long)P.Q * P.K;
    if (n > 0) oat_diff_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, g, y);
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
