/*
 * oat.h -- C ABI of liboat.so: the matched projector pair H / H^T of the
 * interpolation-based discrete-to-discrete imaging model of 3-D optoacoustic
 * tomography (arxiv/paper_1304_2017), as hand-written CUDA kernels for sm_100a.
 *
 * Citations are PAPER.md line numbers (+ equation / algorithm).
 *
 *   H   = D G      projection      (Eq. 11 L116 without H^e; G = Eq. 12 L121 and
 *                                   Appendix Eq. 35-39; D = Eq. 13 L125 / Eq. 3)
 *   H^T = G^T D^T  backprojection  (L168; D^T = Eq. 22; G^T = Eq. 23, Alg. 6)
 *
 * The discretisation implemented is "OAT-DISC v1".
 *
 * Conventions
 *   - units: mm and microseconds.
 *   - volume x: nz*ny*nx fp32, x fastest, voxel n = (iz*ny + iy)*nx + ix (Alg. 6 L601 order);
 *     node (ix,iy,iz) sits at origin + spacing*(ix,iy,iz)             (L203, Eq. 9).
 *   - data y: Q*K fp32, index m = q*K + k, time fastest                (Eq. 5).
 *   - pointers named d_* are DEVICE pointers owned by the caller (e.g. torch tensors);
 *     pointers named h_* are HOST pointers owned by the caller.  The library never frees or
 *     reallocates them.  The geometry handle owns its own device tables and scratch buffers.
 *   - every function returns 0 (OAT_OK) or a negative error code, never throws, never exits;
 *     oat_last_error() gives a thread-local message for the last failure on this thread.
 *   - `cuda_stream` is a cudaStream_t (NULL = the legacy default stream).  Calls are
 *     asynchronous on that stream unless stated otherwise.  One handle must not be used from two
 *     streams at the same time (its scratch buffers are shared).
 *   - there is no CPU fallback: without a CUDA device every call fails with OAT_ERR_CUDA.
 */
#ifndef OAT_H
#define OAT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OAT_OK 0
#define OAT_ERR_INVALID (-1) /* bad argument / descriptor */
#define OAT_ERR_ALLOC (-2)   /* host or device allocation failed */
#define OAT_ERR_CUDA (-3)    /* CUDA runtime error (message has the CUDA string) */

/* Problem statement of the paper: reconstruction cuboid (L203), point-like transducers (L114),
 * speed of sound, first sample time t_min, sampling interval, number of samples (L203, L255). */
typedef struct {
    int32_t nx, ny, nz;      /* nodes per axis (N_x, N_y, N_z), each >= 1 */
    double spacing;          /* Delta_s > 0 */
    double origin[3];        /* (x_min, y_min, z_min): position of node (0,0,0) */
    int32_t n_trans;         /* Q >= 0 */
    const double *trans_xyz; /* HOST, Q x 3 row-major, copied at create */
    double c;                /* c_0 > 0 */
    double t0;               /* t_min >= 0: time of sample k = 0 */
    double dt;               /* Delta_t > 0 */
    int32_t nt;              /* K >= 1 */
    double surf_step;        /* h: surface patch size of Eq. (37); 0 => spacing */
    int32_t kband;           /* B: consecutive time samples sharing one angular rule (reading G11);
                                0 => 32; 1 = the paper's per-sample rule; must be <= 32 */
    double gain;             /* kappa = beta/(4 pi C_p) of Eq. (3); 0 => 1 */
} oat_geometry_desc;

typedef struct oat_geometry oat_geometry;

/* Validates the descriptor (sizes, positive steps, finite positions, no transducer at the grid
 * centre -- the local frame of Appendix L349 is undefined there), computes per-transducer frames
 * and per-band ring tables in fp64 on the host, uploads them to `device`, allocates scratch.
 * *out is set only on success. */
int oat_geometry_create(const oat_geometry_desc *desc, int device, oat_geometry **out);

/* Frees device and host tables.  NULL is a no-op.  The caller must have synchronised its streams. */
void oat_geometry_destroy(oat_geometry *geom);

/* Pure queries (negative on NULL). */
int64_t oat_num_voxels(const oat_geometry *geom);  /* nx*ny*nz */
int64_t oat_num_samples(const oat_geometry *geom); /* Q*K */
/* Number of quadrature samples of OAT-DISC v1 that fall inside the zero-padded node box (the
 * "interpolation samples" of the throughput metric).  Counted on the GPU on first use by a
 * traversal-only kernel (synchronises the device once), then cached. */
int64_t oat_num_surface_samples(oat_geometry *geom);

/* y = H x.  d_x: nz*ny*nx fp32 (read), d_y: Q*K fp32 (OVERWRITTEN).  x and y must not alias. */
int oat_project(oat_geometry *geom, const float *d_x, float *d_y, void *cuda_stream);

/* x = H^T y.  d_y: Q*K fp32 (read), d_x: nz*ny*nx fp32 (OVERWRITTEN; the library zeroes it). */
int oat_backproject(oat_geometry *geom, const float *d_y, float *d_x, void *cuda_stream);

/* Adjoint test: lhs = <Hx, y>, rhs = <x, H^T y> with fp64 reductions on internal scratch,
 * rel = |lhs - rhs| / max(|lhs|, |rhs|).  Synchronises `cuda_stream` before returning. */
int oat_adjoint_check(oat_geometry *geom, const float *d_x, const float *d_y,
                      double *lhs, double *rhs, double *rel, void *cuda_stream);

/* Same operators with HOST buffers: pinned-or-pageable host memory in, host memory out; the
 * host->device and device->host copies are part of the call, which returns after the result has
 * landed in h_y / h_x (used for the end-to-end figure of bench.py). */
int oat_project_host(oat_geometry *geom, const float *h_x, float *h_y);
int oat_backproject_host(oat_geometry *geom, const float *h_y, float *h_x);

/* Row C1: n_iter steps of CGLS (= linear CG on H^T H x = H^T y, L265) from
 * x = 0 with fp32 vectors and fp64 dot products; one H and one H^T per iteration (L273).
 * d_y: Q*K (read), d_x: nz*ny*nx (OVERWRITTEN with the iterate after n_iter steps).
 * h_res / h_grad: HOST arrays of n_iter+1 doubles (may be NULL) receiving ||y - H x_i|| / ||y||
 * and ||H^T (y - H x_i)|| for i = 0..n_iter.  Synchronises the stream every iteration. */
int oat_cgls(oat_geometry *geom, const float *d_y, float *d_x, int n_iter,
             double *h_res, double *h_grad, void *cuda_stream);

/* ---- Row NEXT-1: the electrical impulse response H^e, the smoothness penalty R and the
 * penalised least-squares CG loop "PLS-Int" of the paper (Eq. 29).
 *
 * oat_eir_set: h_he = HOST array of `len` taps [h^e]_m = dt h^e(m dt), m = 0..len-1 (Eq. 14), copied; taps
 * outside that range are zero (reading G20).  len = 0 removes the EIR.  Synchronises the device.
 * oat_eir_apply: adjoint = 0: Eq. (14), d_out[q,k] = sum_kappa h^e[k-1-kappa] d_in[q,kappa];
 *                adjoint = 1: Eq. (21), d_out[q,k] = sum_kappa h^e[kappa-1-k] d_in[q,kappa].
 * Both buffers Q*K fp32 on the device, distinct; d_out is OVERWRITTEN; asynchronous on the stream. */
int oat_eir_set(oat_geometry *geom, const float *h_he, int32_t len);
int oat_eir_apply(oat_geometry *geom, const float *d_in, float *d_out, int adjoint, void *cuda_stream);

/* u = H^e D G x (Eq. 11) and x = G^T D^T H^e† u (L168); without an EIR set they equal oat_project /
 * oat_backproject.  Same buffer rules. */
int oat_project_eir(oat_geometry *geom, const float *d_x, float *d_u, void *cuda_stream);
int oat_backproject_eir(oat_geometry *geom, const float *d_u, float *d_x, void *cuda_stream);

/* Quadratic smoothness penalty, Eq. (34) L305 (reading G21: a voxel on the low face has no neighbour "before" it
 * and that term is omitted).  oat_penalty_apply: d_lx = L x with R(x) = x^T L x (so grad R = 2 L x); volumes
 * nz*ny*nx fp32 on the device, distinct, d_lx OVERWRITTEN, asynchronous.  oat_penalty_value: *value = R(x) with an
 * fp64 reduction; synchronises the stream. */
int oat_penalty_apply(oat_geometry *geom, const float *d_x, float *d_lx, void *cuda_stream);
int oat_penalty_value(oat_geometry *geom, const float *d_x, double *value, void *cuda_stream);

/* ---- Penalty value without any allocation, for callers that cannot call cudaMalloc.
 *
 * Such callers exist: an application that has given all free GPU memory to its own pool (a further cudaMalloc fails or
 * eats into the pool), and a real-time acquisition / reconstruction loop that may not tolerate the device-wide
 * synchronisation every cudaMalloc and cudaFree brings.  oat_penalty_value does not work for them: it needs a geometry
 * handle (creating one allocates) and allocates a volume-sized scratch buffer the first time it runs.
 *
 * oat_penalty_value_noalloc computes the same R(x) = x^T L x (Eq. 34, reading G21) with no handle and no
 * allocation of any kind (no cudaMalloc / cudaFree / cudaMallocHost, no allocating library routine): its scratch -- the
 * fp32 volume L x plus one fp64 accumulator -- is a fixed array inside liboat.so's device image.
 *
 *   nx, ny, nz  nodes per axis, each >= 1, with nx*ny*nz <= OAT_NOALLOC_MAX_VOXELS; a larger volume is refused with
 *               OAT_ERR_INVALID and a message that names the limit (nothing is launched).
 *   d_x         DEVICE, nz*ny*nx fp32, x fastest, owned by the caller, read only; must live on the calling thread's
 *               CURRENT device (checked; host pointers are refused too).
 *   h_value     HOST, one double, owned by the caller; written before the call returns.
 *   cuda_stream a stream of the current device (NULL = legacy default stream).  The work is enqueued there and the call
 *               waits for that stream before returning.
 *
 * Cost of the limit: the array is 8 MiB + 256 B (OAT_NOALLOC_MAX_VOXELS = 2^21 voxels, e.g. 128^3) and every GPU on which
 * this process uses liboat.so carries it until the process exits, whether or not this function is ever called.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress; cached per device afterwards).
 * Make that first call at start-up, before any stream capture begins.
 * Sharing: all calls on one device use the same array, and it keeps what the previous call left.  The function zeroes
 * the accumulator itself and overwrites every element of L x it reads, so back-to-back calls are independent -- but two
 * calls whose GPU work can overlap (different streams, or different host threads) race on the array and return garbage.
 * Serialise them.
 * Result: identical arithmetic to oat_penalty_value (fp32 stencil, fp64 sum); the two agree to the rounding of the
 * fp64 atomic summation order (~1e-15 relative). */
#define OAT_NOALLOC_MAX_VOXELS (1 << 21)
int oat_penalty_value_noalloc(int32_t nx, int32_t ny, int32_t nz, const float *d_x, double *h_value, void *cuda_stream);

/* PLS-Int (Eq. 29; reading G22): n_iter steps of linear CG on (H^T H + mu L) x = H^T u from x = 0 with
 * H = H^e D G (the EIR set by oat_eir_set, if any); one H and one H^T per iteration (L273); fp32 vectors, fp64 dot
 * products.  d_u: Q*K (read), d_x: nz*ny*nx (OVERWRITTEN with the iterate after n_iter steps), mu >= 0.
 * h_obj / h_grad: HOST arrays of n_iter+1 doubles (may be NULL) receiving ||u - H x_i||^2 + mu R(x_i) and
 * ||H^T u - (H^T H + mu L) x_i|| for i = 0..n_iter.  Synchronises the stream every iteration. */
int oat_pls_cg(oat_geometry *geom, const float *d_u, float *d_x, int n_iter, double mu,
               double *h_obj, double *h_grad, void *cuda_stream);

/* ---- Row NEXT-2: filtered backprojection, the discretised FBP formula Eq. (27) L221 (Eq. 4 L69 with Eq. 25-26),
 * voxel driven (Alg. 2), with one weight per transducer (reading G23):
 *   x[n] = sum_q w[q] { (1.5 - (k+tau)/(k~+tau)) p[q,k+1] + ((k+1+tau)/(k~+tau) - 1.5) p[q,k] },
 *   k~ = (|r_q - r_n|/c - t0)/dt, k = floor(k~), tau = t0/dt; pairs with k < 0 or k+1 > K-1 contribute nothing.
 * For the paper's ring/view geometry w[q] = -C_p R^s dtheta dphi sin(theta_q) / (pi beta c^3 dt).
 * d_p: Q*K fp32 pressure data (read), d_w: Q fp32 weights (read), d_x: nz*ny*nx fp32 (OVERWRITTEN); device
 * pointers owned by the caller; asynchronous on the stream. */
int oat_fbp(oat_geometry *geom, const float *d_p, const float *d_w, float *d_x, void *cuda_stream);

/* The weights of Eq. (27) L221 from the patch areas dS_q of the transducers (reading G23):
 *   w[q] = -dS_q / (4 pi^2 kappa c^3 dt R_q),  kappa = the descriptor's gain, R_q = |r_q - grid centre| (L203);
 * for the paper's geometry dS_q = (R^s)^2 dtheta dphi sin(theta_q) gives the printed constant.  h_areas: HOST, Q doubles
 * (read); h_w: HOST, Q floats (written).  No device work. */
int oat_fbp_weights(const oat_geometry *geom, const double *h_areas, float *h_w);

/* ---- Row NEXT-3: the spherical-voxel imaging model in the temporal frequency domain and its adjoint (Eq. 17-20
 * L137-161, Eq. 24; Algs. 7-12), for point-like transducers (Alg. 9 line 7; reading G28).
 * oat_sph_set: frequencies f_l = f0 + l df (MHz), l = 0..nf-1 (reading G27); h_he = HOST array of 2*nf floats, the EIR
 * spectrum h~e(f_l) as (re, im) pairs, or NULL for h~e = 1; p~0(f_l) of Eq. (19) is precomputed (p~0(0) = 0).  nf = 0
 * removes the grid.  Synchronises the device.
 * oat_sph_project:     u[q,l] = p~0(f_l) sum_n x_n exp(-j 2 pi f_l d_qn/c) / (2 pi d_qn)          (Eq. 17-18)
 * oat_sph_backproject: x_n = Re sum_q sum_l u[q,l] conj(p~0(f_l)) exp(+j 2 pi f_l d_qn/c) / (2 pi d_qn)   (Eq. 24; real part:
 *                      reading G29, so that Re<Hx,u> = <x,H†u>)
 * d_x: nz*ny*nx fp32; d_u: Q*nf complex as interleaved (re, im) fp32 pairs, index q*nf + l; device pointers owned by the
 * caller; the output is OVERWRITTEN; asynchronous on the stream. */
int oat_sph_set(oat_geometry *geom, int32_t nf, double f0, double df, const float *h_he);

/* Finite transducer aperture: the spatial impulse response of Eq. (18), (1/S_q) h~_q(r_n, f) = (1/S_q) int_{S_q}
 * exp(-j 2 pi f |r^s - r_n|/c) / (2 pi |r^s - r_n|) dr^s, which the paper names as the reason for this model (L243; its
 * elements are 2 x 2 mm^2, L291).  Reading G30: S_q is a flat square of side `side` (mm) centred on r_q, normal towards
 * the grid centre, sides along the x^tr / y^tr axes of the transducer's frame (Appendix); the integral is the m x m
 * midpoint rule, i.e. the mean of the point responses at the sub-element centres.  side = 0 or m = 1: point-like
 * (the default).  Applies to oat_sph_project / oat_sph_backproject / oat_sph_pls_cg of this handle; cost grows with
 * m^2.  Synchronises the device. */
int oat_sph_set_aperture(oat_geometry *geom, double side, int32_t m);
int oat_sph_project(oat_geometry *geom, const float *d_x, float *d_u, void *cuda_stream);
int oat_sph_backproject(oat_geometry *geom, const float *d_u, float *d_x, void *cuda_stream);

/* PLS-Sph (Eq. 30): the loop of oat_pls_cg with H = H_sph (the grid of oat_sph_set) and its real-part adjoint;
 * d_u: Q*nf complex as interleaved (re, im) fp32 pairs (read), d_x: nz*ny*nx fp32 (OVERWRITTEN), mu >= 0; h_obj / h_grad as
 * in oat_pls_cg with ||.|| the norm of C^{Q nf}.  Synchronises the stream every iteration. */
int oat_sph_pls_cg(oat_geometry *geom, const float *d_u, float *d_x, int n_iter, double mu,
                   double *h_obj, double *h_grad, void *cuda_stream);

/* Number of kernels the last oat_project / oat_backproject on this handle launched. */
int oat_last_launch_count(const oat_geometry *geom);

const char *oat_last_error(void);
const char *oat_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OAT_H */
