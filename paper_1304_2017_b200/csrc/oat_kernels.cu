// Geometry, fallback and vector kernels of liboat.so for sm_100a (B200).  The hot path -- the marching kernels of H and
// H^T -- is in oat_march.cu; the kernels of the NEXT rows (EIR, penalty, FBP, spherical-voxel pair) are in oat_next.cu.
//
// Here: (1) once per geometry: the fp64 direction table, the patch list (generated, culled against the padded box and
// sorted by the Morton code of the patch centre; cub radix sort, a library call made once per geometry); (2) the
// GENERIC patch kernel: warp = one ray, lane = one time sample, 8 scalar loads / atomics per sample on a zero-padded
// linear volume.  It serves bands of fewer than 32 samples and grids the marching kernels cannot index, and it is the
// in-box sample counter (MODE 2); it builds the same rays from the same tables, so all three kernels visit the same
// samples (Eq. 12 vs Eq. 23; Alg. 4 vs Alg. 6); (3) pad / unpad, the adjoint time stencil, the face-quad fold and the
// vector kernels of the CG loops.
#include "oat_internal.h"

#include <math.h>

#include <cub/device/device_radix_sort.cuh>

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

// the 8 corner values of the sample's cell (v[cz*4 + cy*2 + cx]); lanes that are not in the box read
// cell 0 (valid memory) so that the loads of several list entries can be issued back to back
__device__ __forceinline__ void fetch8(const OatDev &P, const float *__restrict__ xpad, const Sample &s, bool in, float v[8])
{
    const int ix = in ? s.ix : 0, iy = in ? s.iy : 0, iz = in ? s.iz : 0;
    const float *p = xpad + (unsigned)((iz * P.py + iy) * P.px + ix);
    v[0] = __ldg(p); v[1] = __ldg(p + 1);
    v[2] = __ldg(p + P.px); v[3] = __ldg(p + P.px + 1);
    const float *p1 = p + P.pxy;
    v[4] = __ldg(p1); v[5] = __ldg(p1 + 1);
    v[6] = __ldg(p1 + P.px); v[7] = __ldg(p1 + P.px + 1);
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
template <int MODE>
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
            for (int u = 0; u < OAT_U; ++u) fetch8(P, xpad, s[u], in[u], v[u]);
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
                if (!in[u]) continue;
                const unsigned idx = (unsigned)((s[u].iz * P.py + s[u].iy) * P.px + s[u].ix);
                const float cw = coef * om[u];
                const float wz1 = s[u].fz * cw, wz0 = cw - wz1;
                const float gx = 1.f - s[u].fx, gy = 1.f - s[u].fy;
                const float w00 = gx * gy, w10 = s[u].fx * gy, w01 = gx * s[u].fy, w11 = s[u].fx * s[u].fy;
                float *p = xacc + idx;                             // Alg. 6: one atomic per corner
                atomicAdd(p, w00 * wz0);
                atomicAdd(p + 1, w10 * wz0);
                atomicAdd(p + P.px, w01 * wz0);
                atomicAdd(p + P.px + 1, w11 * wz0);
                float *p1 = p + P.pxy;
                atomicAdd(p1, w00 * wz1);
                atomicAdd(p1 + 1, w10 * wz1);
                atomicAdd(p1 + P.px, w01 * wz1);
                atomicAdd(p1 + P.px + 1, w11 * wz1);
            }
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
// Work item = PATCH = (q, band, block of OAT_RI rings, azimuth sector): a compact piece of
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

template <int MODE>
__global__ void __launch_bounds__(OAT_NT, 3)
oat_patch_kernel(const OatDev P, const float *__restrict__ xpad, float *__restrict__ xacc,
                 const float *__restrict__ y, double *__restrict__ g, unsigned long long *__restrict__ counter)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Entry *list = reinterpret_cast<Entry *>(smem_raw);
    __shared__ double s_frame[12];
    __shared__ float s_red[OAT_NW][32];
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
            consume_list<MODE>(P, list, s_count, warp, lane, L, xpad, xacc, acc, cnt);
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

// The CG loops keep their scalars on the device (no host round trip per iteration): the vector updates read the step from
// scal[idx] and do nothing when scal[flag] == 0 (a degenerate step: the loop leaves the vectors as they are).
__global__ void oat_axpy_dev_kernel(const double *__restrict__ scal, int idx, int flag, float sign, const float *__restrict__ x,
                                    float *__restrict__ y, long long n)
{
    if (scal[flag] == 0.0) return;
    const float alpha = sign * (float)scal[idx];
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        y[i] = fmaf(alpha, x[i], y[i]);
}

__global__ void oat_xpay_dev_kernel(const float *__restrict__ x, const double *__restrict__ scal, int idx, int flag, float *__restrict__ y, long long n)
{
    if (scal[flag] == 0.0) return;
    const float beta = (float)scal[idx];
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        y[i] = fmaf(beta, y[i], x[i]);
}

// Scalar steps of the CG loops, one thread.  s: [0] gamma = |s|^2 (CGLS) or |r|^2 (PLS), [1] |q|^2 or <p, w>, [2] the new gamma,
// [3] alpha, [4] beta, [5] |r|^2 or |d|^2 (data residual), [6] |y|^2 or the penalty x^T L x, [7] flag: 0 = degenerate step.
// curves (pinned host memory, written through UVA): a[it], b[it].
__global__ void oat_cg_scalar_kernel(double *s, int op, int it, double mu, double *curve_a, double *curve_b)
{
    switch (op) {
    case 0:                                                // CGLS start: curves[0] = (1 or 0, |s|)
        if (curve_a) curve_a[0] = s[6] > 0.0 ? 1.0 : 0.0;
        if (curve_b) curve_b[0] = sqrt(s[0]);
        break;
    case 1:                                                // alpha = gamma / [1]
        s[7] = (s[1] > 0.0 && s[0] > 0.0) ? 1.0 : 0.0;
        s[3] = s[7] != 0.0 ? s[0] / s[1] : 0.0;
        break;
    case 2:                                                // beta = gamma_new / gamma; gamma = gamma_new
        if (s[7] != 0.0) { s[4] = s[2] / s[0]; s[0] = s[2]; }
        break;
    case 3:                                                // CGLS curves of iteration it (after the update)
        if (curve_a) curve_a[it + 1] = s[6] > 0.0 ? sqrt(s[5]) / sqrt(s[6]) : 0.0;
        if (curve_b) curve_b[it + 1] = sqrt(s[0]);
        break;
    case 4:                                                // PLS start: objective |u|^2, gradient |r|
        if (curve_a) curve_a[0] = s[5];
        if (curve_b) curve_b[0] = sqrt(s[0]);
        break;
    case 5:                                                // PLS curves: |d|^2 + mu x^T L x, |r|; a degenerate step repeats the last values
        if (curve_a) curve_a[it + 1] = s[7] != 0.0 ? s[5] + mu * s[6] : curve_a[it];
        if (curve_b) curve_b[it + 1] = s[7] != 0.0 ? sqrt(s[0]) : curve_b[it];
        break;
    }
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

void oat_launch_unface(const OatDev &P, const float4 *faces, float *x, cudaStream_t st)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    oat_unface_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, faces, x);
}

void oat_launch_unpad(const OatDev &P, const float *xpad, float *x, cudaStream_t st)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    oat_unpad_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, xpad, x);
}

template <int MODE>
static cudaError_t launch_patch_t(const OatDev &P, const float *xpad, float *xacc, const float *y, double *g,
                                  unsigned long long *counter, cudaStream_t st)
{
    const size_t smem = sizeof(Entry) * OAT_RI * OAT_RJ;
    // per device: the attribute belongs to the function on the CURRENT device (one process may drive several GPUs)
    cudaError_t e = cudaFuncSetAttribute(oat_patch_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e) return e;
    const long long cap = 0x7fffffffLL;
    const unsigned grid = (unsigned)(P.n_patches < cap ? P.n_patches : cap);
    oat_patch_kernel<MODE><<<grid, OAT_NT, smem, st>>>(P, xpad, xacc, y, g, counter);
    return cudaGetLastError();
}


void oat_launch_dir_table(const OatDev &P, int n_bands, double2 *dir, cudaStream_t st)
{
    if (n_bands > 0) oat_dir_table_kernel<<<dim3(256, (unsigned)n_bands), 128, 0, st>>>(P, dir);
}

cudaError_t oat_launch_patch(int mode, const OatDev &P, const float *xpad, float *xacc, const float *y,
                             double *g, unsigned long long *counter, cudaStream_t st)
{
    if (P.n_patches <= 0) return cudaSuccess;
    if (mode == 0) return launch_patch_t<0>(P, xpad, xacc, y, g, counter, st);
    if (mode == 1) return launch_patch_t<1>(P, xpad, xacc, y, g, counter, st);
    return launch_patch_t<2>(P, xpad, xacc, y, g, counter, st);
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
    // The generator appends patches in whatever order its blocks run.  Two stable radix sorts make the list deterministic:
    // first by the packed descriptor (q, band, ring block, sector), then by the Morton key -- inside a Morton cell the
    // patches are transducer-major, and the order (hence the fp32 summation order of H^T) is the same for every create.
    unsigned long long *vals3 = nullptr;
    OAT_TRY(cudaMalloc((void **)&keys2, sizeof(unsigned) * n));
    OAT_TRY(cudaMalloc((void **)&vals2, sizeof(unsigned long long) * n));
    size_t tmp_bytes = 0, tmp_bytes2 = 0;
    OAT_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, vals, vals2, keys, keys2, (long long)n, 0, 64));
    OAT_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes2, keys2, keys, vals2, vals3, (long long)n, 0, 30));
    if (tmp_bytes2 > tmp_bytes) tmp_bytes = tmp_bytes2;
    OAT_TRY(cudaMalloc(&tmp, tmp_bytes));
    OAT_TRY(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, vals, vals2, keys, keys2, (long long)n, 0, 64));
    cudaError_t e3 = cudaMalloc((void **)&vals3, sizeof(unsigned long long) * n);
    if (e3 != cudaSuccess) { cleanup(); cudaFree(vals2); return e3; }
    e3 = cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys2, keys, vals2, vals3, (long long)n, 0, 30);
    if (e3 == cudaSuccess) e3 = cudaDeviceSynchronize();
    if (e3 != cudaSuccess) { cleanup(); cudaFree(vals2); cudaFree(vals3); return e3; }
    cudaFree(vals2);
    vals2 = vals3;
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

void oat_launch_dot(const float *a, const float *b, long long n, double *out, cudaStream_t st)
{
    if (n > 0) oat_dot_kernel<<<grid_for(n, 256), 256, 0, st>>>(a, b, n, out);
}

void oat_launch_axpy(float alpha, const float *x, float *y, long long n, cudaStream_t st)
{
    if (n > 0) oat_axpy_kernel<<<grid_for(n, 256), 256, 0, st>>>(alpha, x, y, n);
}

void oat_launch_axpy_dev(const double *scal, int idx, int flag, float sign, const float *x, float *y, long long n, cudaStream_t st)
{
    if (n > 0) oat_axpy_dev_kernel<<<grid_for(n, 256), 256, 0, st>>>(scal, idx, flag, sign, x, y, n);
}

void oat_launch_xpay_dev(const float *x, const double *scal, int idx, int flag, float *y, long long n, cudaStream_t st)
{
    if (n > 0) oat_xpay_dev_kernel<<<grid_for(n, 256), 256, 0, st>>>(x, scal, idx, flag, y, n);
}

void oat_launch_cg_scalar(double *scal, int op, int it, double mu, double *curve_a, double *curve_b, cudaStream_t st)
{
    oat_cg_scalar_kernel<<<1, 1, 0, st>>>(scal, op, it, mu, curve_a, curve_b);
}

void oat_launch_xpay(const float *x, float beta, float *y, long long n, cudaStream_t st)
{
    if (n > 0) oat_xpay_kernel<<<grid_for(n, 256), 256, 0, st>>>(x, beta, y, n);
}
