// Kernels of the NEXT rows of SURVEY.md section 8(f) (liboat.so, sm_100a): the electrical impulse response (Eq. 14 / 21),
// the quadratic smoothness penalty (Eq. 34), filtered backprojection (Eq. 27) and the spherical-voxel pair in the
// temporal frequency domain (Eq. 17-19, 24).  None is a dense contraction with a stored operand, so no tensor cores.
#include "oat_internal.h"

#include <math.h>

namespace {


inline int grid_for(long long n, int block)
{
    long long g = (n + block - 1) / block;
    const long long cap = 148LL * 16;                     // grid-stride: a few waves over the 148 SMs
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

// Row NEXT-1, EIR operator.  ADJ = 0: Eq. (14), out[q,k] = sum_m he[m] in[q, k-1-m]; ADJ = 1: Eq. (21),
// out[q,k] = sum_m he[m] in[q, k+1+m]; he[m] given for m = 0..L-1, `in` zero outside [0, K) (reading G20).
// Both are one correlation out[k0+o] = sum_m' h'[m'] win[o + m'] over a window of the row held in shared memory:
//   ADJ = 1: h' = he,           window sample j <-> input k0 + 1 + j
//   ADJ = 0: h'[m'] = he[Lp-1-m'] (taps reversed, Lp = L rounded up to 8 with zero taps), window sample j <-> k0 - Lp + j
// One block = one transducer row x a tile of 2048 outputs; a thread owns 8 CONSECUTIVE outputs and slides a 16-sample
// register window over the taps: per group of 8 taps 64 FMAs against 4 LDS.128 (the one-output-per-thread form needed
// 2 shared-memory loads per FMA and ran at 5 % of the HBM rate).  Every output is one fixed-order fp32 FMA chain
// (deterministic); algorithmic bytes = read + write of the data vector once, algorithmic work = L FMAs per output.
#define OAT_ET 256          // threads per block
#define OAT_ER 8            // outputs per thread
template <int ADJ>
__global__ void __launch_bounds__(OAT_ET)
oat_eir_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ he, int L, int Lp, int K)
{
    extern __shared__ __align__(16) float sm[];
    float *s_h = sm, *s_w = sm + Lp;                       // taps h'[0, Lp), window [0, T + Lp + 8)
    constexpr int T = OAT_ET * OAT_ER;
    const int q = blockIdx.x, k0 = blockIdx.y * T, t = threadIdx.x;      // transducers on grid.x (no 65535 limit on Q)
    const float *row = in + (size_t)q * K;
    for (int m = t; m < Lp; m += OAT_ET) {
        const int src = ADJ ? m : Lp - 1 - m;
        s_h[m] = src < L ? he[src] : 0.f;
    }
    const int base = ADJ ? k0 + 1 : k0 - Lp;
    for (int j = t; j < T + Lp + 8; j += OAT_ET) {
        const int kk = base + j;
        s_w[j] = (kk >= 0 && kk < K) ? row[kk] : 0.f;
    }
    __syncthreads();
    float acc[OAT_ER], x[2 * OAT_ER];
#pragma unroll
    for (int r = 0; r < OAT_ER; ++r) acc[r] = 0.f;
    const float4 *w4 = reinterpret_cast<const float4 *>(s_w + t * OAT_ER);
    const float4 *h4 = reinterpret_cast<const float4 *>(s_h);
    {
        const float4 a = w4[0], b = w4[1];
        x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
    }
    for (int m0 = 0; m0 < Lp; m0 += 8) {
        const float4 a = w4[m0 / 4 + 2], b = w4[m0 / 4 + 3];
        x[8] = a.x; x[9] = a.y; x[10] = a.z; x[11] = a.w; x[12] = b.x; x[13] = b.y; x[14] = b.z; x[15] = b.w;
        const float4 ha = h4[m0 / 4], hb = h4[m0 / 4 + 1];           // same address for the whole block: a broadcast
        const float h[8] = {ha.x, ha.y, ha.z, ha.w, hb.x, hb.y, hb.z, hb.w};
#pragma unroll
        for (int mm = 0; mm < 8; ++mm)
#pragma unroll
            for (int r = 0; r < OAT_ER; ++r) acc[r] = fmaf(h[mm], x[r + mm], acc[r]);
#pragma unroll
        for (int r = 0; r < OAT_ER; ++r) x[r] = x[r + 8];
    }
    const int k = k0 + t * OAT_ER;
    float *o = out + (size_t)q * K + k;
    if (k + OAT_ER <= K && (((size_t)q * K + k) & 3) == 0) {
        reinterpret_cast<float4 *>(o)[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        reinterpret_cast<float4 *>(o)[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
    } else {
#pragma unroll
        for (int r = 0; r < OAT_ER; ++r) if (k + r < K) o[r] = acc[r];
    }
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
            const float rden = ok ? __fdividef(1.f, (float)den) : 0.f;   // a voxel on a transducer: no term at all (reading G25)
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
struct OatSph { int nf, n_lg; double f0, df, ds_over_c, ds; int m; double a_nodes; };   // ds_over_c: microseconds per node unit of distance;
                                                                                   // m x m sub-elements of a square aperture of side a_nodes (node units), reading G30

__global__ void __launch_bounds__(128)
oat_sph_fwd_kernel(const OatDev P, const OatSph S, const float *__restrict__ x, const float2 *__restrict__ p0, float *__restrict__ u)
{
    __shared__ float s_x[OAT_SV];
    const long long n_vox = (long long)P.nx * P.ny * P.nz;
    const long long v0 = (long long)blockIdx.x * OAT_SV;                 // voxel chunks on grid.x: up to 2^31 - 1 of them (the handle allows 2^40 voxels)
    const int nv = (int)min((long long)OAT_SV, n_vox - v0);
    int any = 0;
    for (int i = threadIdx.x; i < nv; i += blockDim.x) { const float v = x[v0 + i]; s_x[i] = v; any |= (v != 0.f); }
    if (!__syncthreads_or(any)) return;                    // an all-zero chunk contributes nothing
    const long long wi = (long long)blockIdx.y * blockDim.x + threadIdx.x;
    if (wi >= (long long)P.Q * S.n_lg) return;
    const int q = (int)(wi / S.n_lg), lg = (int)(wi % S.n_lg);
    const int l0 = lg * OAT_SG;
    const double *f = P.frame + (size_t)q * 12;
    const double tx = f[9] - 1.0, ty = f[10] - 1.0, tz = f[11] - 1.0;       // node coordinates (frames hold padded ones)
    // finite aperture (Eq. 18, reading G30): the m x m sub-element midpoints t + u_i A e_x + u_j A e_y, u = (i + 1/2)/m - 1/2
    const double Ax = S.a_nodes * f[0], Ay = S.a_nodes * f[1], Az = S.a_nodes * f[2];
    const double Bx = S.a_nodes * f[3], By = S.a_nodes * f[4], Bz = S.a_nodes * f[5];
    const int m = S.m;
    const double rm = 1.0 / (double)m;
    const float wsub = (float)(rm * rm);                                    // (1/S_q) x sub-element area
    const double fa = S.f0 + (double)l0 * S.df;
    float ar[OAT_SG], ai[OAT_SG];
#pragma unroll
    for (int j = 0; j < OAT_SG; ++j) ar[j] = ai[j] = 0.f;
    int ix = (int)(v0 % P.nx), iy = (int)((v0 / P.nx) % P.ny), iz = (int)(v0 / ((long long)P.nx * P.ny));
    for (int i = 0; i < nv; ++i) {
        const float xv = s_x[i];                           // same address for the whole block: a broadcast
        if (xv != 0.f) {                                   // block-uniform branch
            for (int si = 0; si < m; ++si) {
                const double ui = ((double)si + 0.5) * rm - 0.5;
                for (int sj = 0; sj < m; ++sj) {
                    const double uj = ((double)sj + 0.5) * rm - 0.5;
                    const double dx = (double)ix - (tx + ui * Ax + uj * Bx), dy = (double)iy - (ty + ui * Ay + uj * By),
                                 dz = (double)iz - (tz + ui * Az + uj * Bz);
                    const double d = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
                    if (d > 0.0) {
                        const double td = d * S.ds_over_c;         // |r^s - r_n| / c
                        const double pa = fa * td, pd = S.df * td; // cycles
                        float sr, cr, sz, cz;
                        sincospif((float)(-2.0 * (pa - rint(pa))), &sr, &cr);
                        sincospif((float)(-2.0 * (pd - rint(pd))), &sz, &cz);
                        const float amp = xv * wsub / (float)(6.283185307179586 * d * S.ds);
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
    __shared__ double s_t[OAT_SQ][9];                     // per staged transducer: position, A e_x, A e_y (node units)
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
            if (threadIdx.x < nq * 9) {
                const int j = threadIdx.x / 9, c = threadIdx.x % 9;
                const double *fr = P.frame + (size_t)(q0 + j) * 12;
                s_t[j][c] = c < 3 ? fr[9 + c] - 1.0 : S.a_nodes * fr[c - 3];
            }
            __syncthreads();
            if (!inside) continue;
            const int m = S.m;
            const double rm = 1.0 / (double)m;
            for (int j = 0; j < nq; ++j) {
                for (int sub = 0; sub < m * m; ++sub) {    // sub-elements of the aperture (reading G30); m = 1: the point-like model
                    const double ui = ((double)(sub / m) + 0.5) * rm - 0.5, uj = ((double)(sub % m) + 0.5) * rm - 0.5;
                    const double dx = (double)ix - (s_t[j][0] + ui * s_t[j][3] + uj * s_t[j][6]),
                                 dy = (double)iy - (s_t[j][1] + ui * s_t[j][4] + uj * s_t[j][7]),
                                 dz = (double)iz - (s_t[j][2] + ui * s_t[j][5] + uj * s_t[j][8]);
                    const double d = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
                    if (!(d > 0.0)) continue;
                    const double td = d * S.ds_over_c, pd = S.df * td;
                    float sz, cz;
                    sincospif((float)(2.0 * (pd - rint(pd))), &sz, &cz);
                    const float amp = (float)(rm * rm) / (float)(6.283185307179586 * d * S.ds);
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
    }
    if (inside) x[n] = (float)total;
}

}  // namespace


cudaError_t oat_launch_eir(int adjoint, const float *in, float *out, const float *he, int L, int Q, int K, cudaStream_t st)
{
    if (Q <= 0 || K <= 0) return cudaSuccess;
    const int Lp = ((L + 7) / 8) * 8, T = OAT_ET * OAT_ER;
    const size_t smem = sizeof(float) * (size_t)(2 * Lp + T + 8);
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(oat_eir_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(oat_eir_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const dim3 grid((unsigned)Q, (unsigned)((K + T - 1) / T));            // grid.y <= 65535 holds for K < 1.3e8 (K is an int32 count of 2048-sample chunks)
    if (grid.y > 65535u) return cudaErrorInvalidValue;
    if (adjoint) oat_eir_kernel<1><<<grid, OAT_ET, smem, st>>>(in, out, he, L, Lp, K);
    else oat_eir_kernel<0><<<grid, OAT_ET, smem, st>>>(in, out, he, L, Lp, K);
    return cudaGetLastError();
}

void oat_launch_fbp(const OatDev &P, const float *p, const float *wq, float *x, cudaStream_t st)
{
    const dim3 grid((unsigned)((P.nx + 7) / 8), (unsigned)((P.ny + 7) / 8), (unsigned)((P.nz + 3) / 4));
    oat_fbp_kernel<<<grid, 256, 0, st>>>(P, p, wq, x);
}

cudaError_t oat_launch_sph_fwd(const OatDev &P, int nf, double f0, double df, double ds, double c, double aperture, int m, const float *x, const float2 *p0, float *u, cudaStream_t st)
{
    OatSph S; S.nf = nf; S.n_lg = (nf + OAT_SG - 1) / OAT_SG; S.f0 = f0; S.df = df; S.ds = ds; S.ds_over_c = ds / c;
    S.m = (aperture > 0.0 && m > 1) ? m : 1; S.a_nodes = S.m > 1 ? aperture / ds : 0.0;
    const long long n_vox = (long long)P.nx * P.ny * P.nz, work = (long long)P.Q * S.n_lg;
    if (n_vox <= 0 || work <= 0) return cudaSuccess;
    const long long gx = (n_vox + OAT_SV - 1) / OAT_SV, gy = (work + 127) / 128;
    if (gx > 2147483647LL || gy > 65535LL) return cudaErrorInvalidValue;          // > 8.4e6 (transducer, frequency group) pairs
    const dim3 grid((unsigned)gx, (unsigned)gy);
    oat_sph_fwd_kernel<<<grid, 128, 0, st>>>(P, S, x, p0, u);
    return cudaGetLastError();
}

void oat_launch_sph_bwd(const OatDev &P, int nf, double f0, double df, double ds, double c, double aperture, int m, const float2 *u, const float2 *p0, float2 *v, float *x, cudaStream_t st)
{
    OatSph S; S.nf = nf; S.n_lg = (nf + OAT_SG - 1) / OAT_SG; S.f0 = f0; S.df = df; S.ds = ds; S.ds_over_c = ds / c;
    S.m = (aperture > 0.0 && m > 1) ? m : 1; S.a_nodes = S.m > 1 ? aperture / ds : 0.0;
    const long long n_vox = (long long)P.nx * P.ny * P.nz, n = (long long)P.Q * nf;
    if (n > 0) oat_sph_prep_kernel<<<grid_for(n, 256), 256, 0, st>>>(S, P.Q, u, p0, v);
    if (n_vox > 0) oat_sph_bwd_kernel<<<(unsigned)((n_vox + 127) / 128), 128, 0, st>>>(P, S, v, x);
}

void oat_launch_penalty(const OatDev &P, const float *x, float *out, float alpha, float beta, cudaStream_t st)
{
    const long long n = (long long)P.nx * P.ny * P.nz;
    if (n > 0) oat_penalty_kernel<<<grid_for(n, 256), 256, 0, st>>>(P, x, out, alpha, beta);
}
