// Internal declarations of liboat.so (not part of the C ABI; see include/oat.h).
//
// Data layout in HBM:
//   frame   Q x 12 fp64   e_x, e_y, e_z (Appendix, reading S1) and base' = (r_q - o)/ds + 1,
//                         the transducer position in PADDED fractional node coordinates
//   band    NB            per band of B time samples: reference radius, dtheta, ring-table slice
//   ring    sum(n_rings+1) per band, rings i = 1..n_rings with theta_i = i*dtheta < pi, plus a
//                         sentinel whose `cum` is the band's total direction count
//   qb_rings Q x NB       number of leading rings that can reach the padded box (S9 cull)
//   patches               Morton-sorted work items (q, band, ring block, azimuth sector)
//   dir                   fp64 direction table of the marching kernels
//   cells                 per-cell polynomial records with a zero margin (marching H)
//   faces                 face-quad accumulators of the three orientations (marching H^T)
//   xpad    (nz+2)(ny+2)(px) fp32  volume zero-padded by one node on every side = Eq. (12)'s
//                         "nodes outside the grid do not exist" (reading G5), row pitch px (generic kernel)
//   g       Q x K fp64    SRT accumulator (forward) before the time difference
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define OAT_NT 256         // threads per block of the generic patch kernel
#define OAT_NW (OAT_NT / 32)
#define OAT_RI 32          // rings per patch
#define OAT_RJ 32          // max azimuth samples per ring of a patch
#define OAT_MT 128         // threads per block of the marching kernels
#define OAT_BU 4           // steps per trip of the (rolled) backprojection marching loop

struct OatBand {
    double s_mid;      // radius of the band's anchor (k0 + (B-1)/2) in voxel units: rho/ds
    double dtheta;     // h / rho_ref (Eq. 37), rho_ref = radius of the band's last sample (S2)
    float s_lo, s_hi;  // radii (voxel units) of the first / last sample with rho > 0
    int ring_ofs;      // first ring of this band in the ring table
    int n_rings;       // rings with theta_i < pi
    int k0, nk;        // first sample and number of samples (ragged last band: nk < B)
    int rb_ofs;        // first entry of this band in the ring-block sector table
    int dir_rings;     // leading rings of this band covered by the direction table (max over q of qb_rings)
    long long dir_ofs; // first direction of this band in the direction table
};

struct __align__(16) OatRing {
    double st, ct;     // sin(theta_i), cos(theta_i)
    float omega;       // solid-angle weight sin(theta_i) dtheta dphi_i (S2)
    int N;             // azimuth count N_{b,i} = max(1, ceil(2 pi rho_ref sin(theta_i) / h))
    int cum;           // directions in rings before this one
    int pad;
};

struct OatDev {
    int nx, ny, nz;            // nodes
    int px, py, pz;            // padded dims: px = row pitch >= nx+2, py = ny+2, pz = nz+2
    long long pxy;             // px*py
    int Q, K, B, NB;
    double c, t0, dt, kappa;
    double step;               // c*dt/ds: voxels per time sample along a ray
    const double *frame;
    const OatBand *band;
    const OatRing *ring;
    const int *qb_rings;
    const int *rb_sectors;               // per (band, ring block): number of azimuth sectors S
    const unsigned long long *patches;   // Morton-sorted packed (q, band, ring block, sector)
    long long n_patches;
    const double2 *dir;                  // direction table (marching kernels): (sin th cos phi, sin th sin phi) of ring r,
                                         // azimuth j of band b at band.dir_ofs + ring.cum + j, fp64 (S2, S3)
    long long max_band_dirs;             // largest number of table directions of one band (the tile kernels pack it into 27 bits)
    const int *q_count;                  // patches per transducer
    int *q_done;                         // patches finished in the running projection (zeroed per call)
    int cx, cy, cz;            // cell-record layout (marching H): cells per row (pitch, multiple of 4) / rows per plane / planes,
    int cm;                    // each = nodes + 1 + 2 cm: a zero margin of cm cells around the padded box, wide enough for every
                               // sample of every ray whose segment meets the box (no per-sample bounds test)
    long long cxy;             // cx*cy; record of padded cell (ix,iy,iz) = ((iz+cm)*cy + iy+cm)*cx + ix+cm, 32 B each
    // face-quad accumulators (marching H^T): orientation o = axis a normal to the quad, in-plane axes
    // (b, c) = (y,z), (z,x), (x,y) for a = x, y, z; record (ia, ib, ic) = float4 of padded nodes
    // {(ib,ic),(ib+1,ic),(ib,ic+1),(ib+1,ic+1)} on plane ia, at f_base[o] + (ia*f_nc[o] + ic)*f_nb[o] + ib
    long long f_base[3];
    int f_nb[3], f_nc[3];
};

// error reporting shared by the translation units (oat_api.cu): formats the thread-local message, returns `code`
int oat_fail(int code, const char *fmt, ...);

// launchers; all asynchronous on `st`
void oat_launch_pad(const OatDev &P, const float *x, float *xpad, cudaStream_t st);
void oat_launch_unpad(const OatDev &P, const float *xpad, float *x, cudaStream_t st);
// generic patch kernel (oat_kernels.cu): mode 0: g += G x (gathers from xpad) and y rows (step A4); 1: xacc += G^T D^T y
// (8 scalar atomics per sample); 2: count in-box samples
cudaError_t oat_launch_patch(int mode, const OatDev &P, const float *xpad, float *xacc, const float *y,
                             double *g, unsigned long long *counter, cudaStream_t st);
// cell records (marching H): per cell the 8 coefficients of its trilinear polynomial
// c0 + c1 fx + c2 fy + c3 fx fy + fz (c4 + c5 fx + c6 fy + c7 fx fy), fp64-computed, one 32-byte sector
void oat_launch_pad_cells(const OatDev &P, const float *x, float4 *cells, cudaStream_t st);
// x[n] = sum of the 12 face-quad components that are node n (marching H^T)
void oat_launch_unface(const OatDev &P, const float4 *faces, float *x, cudaStream_t st);
// marching kernels (oat_march.cu, B = 32): mode 0 gathers from cell records into g (and writes y rows, step A4),
// mode 1 reads the data y_in, forms g'_k rho_k^2 per band at load (step B1) and scatters it into the face-quad accumulators
cudaError_t oat_launch_march(int mode, const OatDev &P, const float4 *cells, float4 *faces, float *y_out,
                             const float *y_in, double *g, cudaStream_t st);
// tile-stationary projection kernel (oat_tile.cu): a block keeps a brick of the volume in shared memory (TMA box load) and evaluates every
// sample that falls into it; needs B = 32, the direction table and 7 c dt < 3 spacing
bool oat_tile_supported(const OatDev &P);
cudaError_t oat_launch_tile_fwd(const OatDev &P, const float *x, double *g, float *y, unsigned long long *counter,
                                unsigned long long *stats, int nq_per_item, int allow_tma, cudaStream_t st);
void oat_launch_dir_table(const OatDev &P, int n_bands, double2 *dir, cudaStream_t st);
cudaError_t oat_build_patches(const OatDev &P, unsigned long long cap, int shift, int *q_count, unsigned long long **patches_out, long long *n_patches);
// vector kernels (row C1 and the adjoint check); dots accumulate in fp64 into *out (pre-zeroed)
void oat_launch_dot(const float *a, const float *b, long long n, double *out, cudaStream_t st);
void oat_launch_axpy(float alpha, const float *x, float *y, long long n, cudaStream_t st);   // y += alpha x
void oat_launch_xpay(const float *x, float beta, float *y, long long n, cudaStream_t st);    // y = x + beta y
// device-scalar forms for the CG loops: y += sign * scal[idx] x, y = x + scal[idx] y (both no-ops when scal[flag] == 0), and the
// one-thread scalar steps (op codes in oat_kernels.cu); curves point to pinned host memory
void oat_launch_axpy_dev(const double *scal, int idx, int flag, float sign, const float *x, float *y, long long n, cudaStream_t st);
void oat_launch_xpay_dev(const float *x, const double *scal, int idx, int flag, float *y, long long n, cudaStream_t st);
void oat_launch_cg_scalar(double *scal, int op, int it, double mu, double *curve_a, double *curve_b, cudaStream_t st);
// row NEXT-1 (oat_next.cu): EIR convolution / correlation along time (Eq. 14 / Eq. 21) and the penalty stencil (Eq. 34)
cudaError_t oat_launch_eir(int adjoint, const float *in, float *out, const float *he, int L, int Q, int K, cudaStream_t st);
void oat_launch_penalty(const OatDev &P, const float *x, float *out, float alpha, float beta, cudaStream_t st);   // out = beta out + alpha L x
// row NEXT-2: filtered backprojection, Eq. (27), x[n] = sum_q wq[q] {...} (voxel driven)
void oat_launch_fbp(const OatDev &P, const float *p, const float *wq, float *x, cudaStream_t st);
// row NEXT-3: spherical-voxel model (Eq. 17-19, 24); point-like transducers or square apertures of side `aperture` (mm)
// integrated with m x m sub-elements (Eq. 18, reading G30); u, v: Q x nf complex (float2), p0: nf complex
cudaError_t oat_launch_sph_fwd(const OatDev &P, int nf, double f0, double df, double ds, double c, double aperture, int m, const float *x, const float2 *p0, float *u, cudaStream_t st);
void oat_launch_sph_bwd(const OatDev &P, int nf, double f0, double df, double ds, double c, double aperture, int m, const float2 *u, const float2 *p0, float2 *v, float *x, cudaStream_t st);
