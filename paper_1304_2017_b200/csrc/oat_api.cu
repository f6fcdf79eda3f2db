// C ABI of liboat.so (include/oat.h): descriptor validation, host fp64 pre-computation of
// per-transducer frames and per-band ring tables (step A1 of SURVEY.md §8(a)), scratch
// management, and the operator entry points.  All hot work is in oat_kernels.cu.
#include "../../include/oat.h"
#include "../../include/oat_probe.h"
#include "oat_internal.h"

#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>
#include <vector>

namespace {

thread_local char g_err[512] = "";

#define fail oat_fail

#define CUDA_TRY(expr)                                                                          \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? OAT_ERR_ALLOC : OAT_ERR_CUDA,         \
                        "%s failed: %s", #expr, cudaGetErrorString(e_));                        \
    } while (0)

const double kPi = 3.14159265358979323846;

}  // namespace

int oat_fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

struct oat_geometry {
    oat_geometry_desc desc;
    int device = 0;
    double h = 0, kappa = 1;
    OatDev dev;                               // kernel parameter block (device pointers inside)
    // device tables
    double *d_frame = nullptr;
    OatBand *d_band = nullptr;
    OatRing *d_ring = nullptr;
    int *d_qb_rings = nullptr;
    int *d_rb_sectors = nullptr;
    unsigned long long *d_patches = nullptr;  // Morton-sorted work items (lazy)
    int *d_q_count = nullptr, *d_q_done = nullptr;
    unsigned long long patch_cap = 0;
    int morton_shift = 6;                     // patches are sorted by the Morton code of (centre >> shift): 64-voxel cells (measured best of 2..10)
    // scratch
    float *d_xpad = nullptr;                  // padded volume (generic kernel: gather source / scatter target; lazy)
    double2 *d_dir = nullptr;                 // direction table of the marching kernels
    float4 *d_faces = nullptr;                // face-quad accumulators of the 3 orientations (marching H^T, lazy)
    size_t n_faces = 0;                       // float4 records, 0 = marching H^T unavailable for this grid
    float4 *d_cells = nullptr;                // per-cell polynomial records (marching H, lazy)
    size_t n_cells = 0;                       // records incl. the zero margin (2 float4 each)
    double *d_g = nullptr;                    // Q*K SRT accumulator
    float *d_y2 = nullptr, *d_x2 = nullptr;   // adjoint check / CGLS / host entry points (lazy)
    float *d_x3 = nullptr, *d_y3 = nullptr, *d_x4 = nullptr;   // CGLS vectors (lazy)
    float *d_y4 = nullptr;                    // EIR scratch (row NEXT-1, lazy)
    float *d_he = nullptr;                    // EIR taps [h^e]_m, m = 0..n_he-1 (Eq. 14), NULL = no EIR
    int n_he = 0;
    float2 *d_p0 = nullptr, *d_sv = nullptr;  // row NEXT-3: p~0(f_l) (Eq. 19) and the scratch v = u conj(p~0)
    float *d_sd = nullptr, *d_sq = nullptr;   // PLS-Sph data-space vectors (2*Q*nf floats, lazy; freed with the grid)
    int sph_nf = 0;
    double sph_f0 = 0, sph_df = 0;
    double sph_aperture = 0;                  // side of the square transducer surface (mm), 0 = point-like (reading G30)
    int sph_m = 1;                            // sub-elements per side of the aperture quadrature
    double *d_scal = nullptr;                 // a few fp64 scalars (dots)
    unsigned long long *d_counter = nullptr;
    double *h_scal = nullptr;                 // pinned mirror of d_scal
    long long n_surface_samples = -1;
    int variant_project = 4, variant_backproject = 4;   // 4 = marching kernels, 0 = generic patch kernel (oat_probe.h)
    int tile_tma = 1;                         // 0: the tile kernels stage the brick with plain loads instead of TMA (measurement aid)
    int tile_nq = 1024;                       // transducers per (tile, transducer range) item of the tile-stationary projection
    unsigned long long *d_tile_stats = nullptr;   // enumeration counters of the tile kernels (oat_probe.h), NULL = off
    bool march_ok = false;                    // ray anchors fit the 10-bit packed offsets of the marching H^T queue, step <= 1
    size_t record_limit = (size_t)1 << 31;    // the marching kernels index records with 32 bits (lowered only by tests)
    int last_launches = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool ev_valid = false;
    size_t n_vox = 0, n_dat = 0, n_pad = 0;
    std::vector<double> h_rq;                 // |r_q - grid centre| per transducer (mm), for oat_fbp_weights
};

namespace {

void free_all(oat_geometry *g)
{
    if (!g) return;
    cudaFree(g->d_frame); cudaFree(g->d_band); cudaFree(g->d_ring); cudaFree(g->d_qb_rings);
    cudaFree(g->d_xpad); cudaFree(g->d_g); cudaFree(g->d_y2);
    cudaFree(g->d_x2); cudaFree(g->d_x3); cudaFree(g->d_y3); cudaFree(g->d_x4); cudaFree(g->d_scal);
    cudaFree(g->d_y4); cudaFree(g->d_he); cudaFree(g->d_p0); cudaFree(g->d_sv); cudaFree(g->d_sd); cudaFree(g->d_sq);
    cudaFree(g->d_counter); cudaFree(g->d_cells); cudaFree(g->d_faces); cudaFree(g->d_dir); cudaFree(g->d_rb_sectors); cudaFree(g->d_patches); cudaFree(g->d_q_count); cudaFree(g->d_q_done); cudaFree(g->d_tile_stats);
    if (g->h_scal) cudaFreeHost(g->h_scal);
    if (g->ev0) cudaEventDestroy(g->ev0);
    if (g->ev1) cudaEventDestroy(g->ev1);
    delete g;
}

// Largest polar angle (about the axis transducer -> grid centre) at which a ray segment with
// radius in [ra, rb] can meet the ball of radius R around the centre at distance L (S9; the paper's
// theta'_max, Alg. 4, extended to a radius interval).  < 0: cannot meet.
double band_theta_max(double L, double R, double ra, double rb)
{
    if (ra >= L + R || rb <= L - R) return -1.0;
    if (ra <= R - L) return kPi;                          // a shell lies wholly inside the ball
    // cos(theta_max(rho)) = f(rho) = (L^2 + rho^2 - R^2) / (2 rho L); minimise f over [ra, rb]
    double rs = ra;
    if (L > R) { rs = sqrt(L * L - R * R); if (rs < ra) rs = ra; if (rs > rb) rs = rb; }
    const double cm = (L * L + rs * rs - R * R) / (2.0 * rs * L);
    if (cm >= 1.0) return -1.0;
    if (cm <= -1.0) return kPi;
    return acos(cm);
}

template <class T>
int upload(T **dst, const std::vector<T> &src)
{
    const size_t bytes = sizeof(T) * (src.size() ? src.size() : 1);
    CUDA_TRY(cudaMalloc((void **)dst, bytes));
    if (!src.empty()) CUDA_TRY(cudaMemcpy(*dst, src.data(), sizeof(T) * src.size(), cudaMemcpyHostToDevice));
    return OAT_OK;
}

int ensure(float **p, size_t n)
{
    if (*p) return OAT_OK;
    CUDA_TRY(cudaMalloc((void **)p, sizeof(float) * (n ? n : 1)));
    return OAT_OK;
}

int build_geometry(oat_geometry *G)
{
    const oat_geometry_desc &d = G->desc;
    const int B = d.kband > 0 ? d.kband : 32;
    const int K = d.nt, Q = d.n_trans;
    const int NB = (K + B - 1) / B;
    G->h = d.surf_step > 0 ? d.surf_step : d.spacing;
    G->kappa = d.gain != 0 ? d.gain : 1.0;
    const double ds = d.spacing, h = G->h;
    const int n[3] = {d.nx, d.ny, d.nz};
    double C[3], r2 = 0;
    for (int a = 0; a < 3; ++a) {
        C[a] = d.origin[a] + ds * 0.5 * (n[a] - 1);
        const double half = ds * (0.5 * (n[a] - 1) + 1.0);
        r2 += half * half;
    }
    const double r_pad = sqrt(r2);

    // ---- bands and rings (S2), fp64, same closed-form rule as the oracle (reading G19)
    std::vector<OatBand> bands(NB);
    std::vector<OatRing> rings;
    for (int b = 0; b < NB; ++b) {
        OatBand &bd = bands[b];
        bd.k0 = b * B;
        bd.nk = (K - bd.k0 < B) ? K - bd.k0 : B;
        const int kref = bd.k0 + bd.nk - 1;
        const double rho_ref = d.c * (d.t0 + kref * d.dt);
        bd.s_mid = d.c * (d.t0 + (bd.k0 + 0.5 * (B - 1)) * d.dt) / ds;
        bd.ring_ofs = (int)rings.size();
        bd.n_rings = 0;
        bd.dtheta = 0;
        int kfirst = bd.k0;                                // first sample with rho > 0
        while (kfirst <= kref && !(d.c * (d.t0 + kfirst * d.dt) > 0)) ++kfirst;
        bd.s_lo = (float)(d.c * (d.t0 + kfirst * d.dt) / ds);
        bd.s_hi = (float)(rho_ref / ds);
        long long cum = 0;
        if (rho_ref > 0 && kfirst <= kref) {
            const double dtheta = h / rho_ref;             // Eq. 37
            bd.dtheta = dtheta;
            for (int i = 1;; ++i) {
                const double theta = i * dtheta;           // Eq. 38
                if (!(theta < kPi)) break;
                OatRing r;
                r.st = sin(theta);
                r.ct = cos(theta);
                double Nd = ceil(2.0 * kPi * rho_ref * r.st / h);
                if (Nd < 1) Nd = 1;
                if (cum + (long long)Nd > 0x7fffffffLL) return fail(OAT_ERR_INVALID, "too many directions in one band (surf_step too small)");
                r.N = (int)Nd;
                r.omega = (float)(r.st * dtheta * (2.0 * kPi / Nd));
                r.cum = (int)cum;
                r.pad = 0;
                cum += r.N;
                rings.push_back(r);
                ++bd.n_rings;
            }
        }
        OatRing sentinel;
        sentinel.st = 0; sentinel.ct = 1; sentinel.omega = 0; sentinel.N = 1; sentinel.cum = (int)cum; sentinel.pad = 0;
        rings.push_back(sentinel);
    }

    // ---- ring blocks of OAT_RI rings and their azimuth sector counts (patches)
    std::vector<int> rb_sectors;
    std::vector<std::vector<long long>> rb_prefix(NB);     // per band: sectors in ring blocks [0, rb)
    for (int b = 0; b < NB; ++b) {
        OatBand &bd = bands[b];
        bd.rb_ofs = (int)rb_sectors.size();
        bd.dir_rings = 0; bd.dir_ofs = 0;
        const int n_rb = (bd.n_rings + OAT_RI - 1) / OAT_RI;
        rb_prefix[b].assign(n_rb + 1, 0);
        for (int rb = 0; rb < n_rb; ++rb) {
            int nmax = 1;
            for (int r = rb * OAT_RI; r < bd.n_rings && r < (rb + 1) * OAT_RI; ++r)
                if (rings[bd.ring_ofs + r].N > nmax) nmax = rings[bd.ring_ofs + r].N;
            const int S = (nmax + OAT_RJ - 1) / OAT_RJ;
            if (S > 0xffff || n_rb > 0x3ff) return fail(OAT_ERR_INVALID, "too many patch sectors / ring blocks (surf_step too small)");
            rb_sectors.push_back(S);
            rb_prefix[b][rb + 1] = rb_prefix[b][rb] + S;
        }
        if (n_rb == 0) rb_sectors.push_back(1);
    }
    if (Q >= (1 << 26) || NB > 0xfff) return fail(OAT_ERR_INVALID, "too many transducers / bands");

    // ---- frames (S1) and the per-(q, band) ring bound (S9)
    std::vector<double> frame((size_t)Q * 12);
    std::vector<int> qb_rings((size_t)Q * NB);
    for (int q = 0; q < Q; ++q) {
        const double *rq = d.trans_xyz + 3 * (size_t)q;
        double v[3] = {C[0] - rq[0], C[1] - rq[1], C[2] - rq[2]};
        const double L = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        if (!(L > 0) || !isfinite(L)) return fail(OAT_ERR_INVALID, "transducer %d is at the grid centre or not finite", q);
        G->h_rq.push_back(L);
        double ez[3] = {v[0] / L, v[1] / L, v[2] / L};
        double ey[3] = {ez[1], -ez[0], 0.0};               // e_z x z^
        const double an = sqrt(ey[0] * ey[0] + ey[1] * ey[1]);
        if (an < 1e-12) { ey[0] = 0; ey[1] = 1; ey[2] = 0; }
        else { ey[0] /= an; ey[1] /= an; }
        const double ex[3] = {ey[1] * ez[2] - ey[2] * ez[1], ey[2] * ez[0] - ey[0] * ez[2], ey[0] * ez[1] - ey[1] * ez[0]};
        double *f = &frame[(size_t)q * 12];
        for (int a = 0; a < 3; ++a) {
            f[a] = ex[a]; f[3 + a] = ey[a]; f[6 + a] = ez[a];
            f[9 + a] = (rq[a] - d.origin[a]) / ds + 1.0;   // padded fractional node coordinates
        }
        for (int b = 0; b < NB; ++b) {
            const OatBand &bd = bands[b];
            int nr = 0;
            if (bd.n_rings > 0) {
                const double th = band_theta_max(L, r_pad, (double)bd.s_lo * ds * (1 - 1e-6), (double)bd.s_hi * ds * (1 + 1e-6));
                if (th >= 0) {
                    const double cnt = floor(th / bd.dtheta) + 1.0;     // rings with theta_i <= th, +1 margin
                    nr = cnt < bd.n_rings ? (int)cnt : bd.n_rings;
                }
            }
            qb_rings[(size_t)q * NB + b] = nr;
            if (nr > 0) G->patch_cap += (unsigned long long)rb_prefix[b][(nr + OAT_RI - 1) / OAT_RI];
        }
    }
    // direction table of the marching kernels: per band the leading rings any transducer can use
    long long n_dir = 0, max_band_dirs = 0;
    for (int b = 0; b < NB; ++b) {
        int mr = 0;
        for (int q = 0; q < Q; ++q) if (qb_rings[(size_t)q * NB + b] > mr) mr = qb_rings[(size_t)q * NB + b];
        bands[b].dir_rings = mr;
        bands[b].dir_ofs = n_dir;
        n_dir += rings[bands[b].ring_ofs + mr].cum;
        if (rings[bands[b].ring_ofs + mr].cum > max_band_dirs) max_band_dirs = rings[bands[b].ring_ofs + mr].cum;
    }

    // ---- upload
    int rc;
    if ((rc = upload(&G->d_frame, frame))) return rc;
    if ((rc = upload(&G->d_band, bands))) return rc;
    if ((rc = upload(&G->d_ring, rings))) return rc;
    if ((rc = upload(&G->d_qb_rings, qb_rings))) return rc;
    if ((rc = upload(&G->d_rb_sectors, rb_sectors))) return rc;

    OatDev &P = G->dev;
    P.nx = d.nx; P.ny = d.ny; P.nz = d.nz;
    P.px = ((d.nx + 2 + 7) / 8) * 8;                       // rows start on 32-byte sectors
    P.py = d.ny + 2; P.pz = d.nz + 2;
    P.pxy = (long long)P.px * P.py;
    P.Q = Q; P.K = K; P.B = B; P.NB = NB;
    P.c = d.c; P.t0 = d.t0; P.dt = d.dt; P.kappa = G->kappa;
    P.step = d.c * d.dt / ds;
    P.frame = G->d_frame; P.band = G->d_band; P.ring = G->d_ring;
    P.qb_rings = G->d_qb_rings;
    P.rb_sectors = G->d_rb_sectors; P.patches = nullptr; P.n_patches = 0;
    P.q_count = nullptr; P.q_done = nullptr;
    P.dir = nullptr;
    P.max_band_dirs = max_band_dirs;
    if (B == 32 && n_dir > 0 && n_dir < (1LL << 31)) {     // 16 B per direction; otherwise the generic kernel is used
        CUDA_TRY(cudaMalloc((void **)&G->d_dir, sizeof(double2) * (size_t)n_dir));
        P.dir = G->d_dir;
    }
    // cell records with a zero margin: a ray is kept when the bounding box of its 32-sample segment meets the padded box,
    // so its samples lie within 31 * step cells of it (+ the cull's 0.01 slack and one cell for floor)
    P.cm = (int)ceil(31.0 * P.step) + 3;
    P.cx = ((d.nx + 1 + 2 * P.cm + 3) / 4) * 4; P.cy = d.ny + 1 + 2 * P.cm; P.cz = d.nz + 1 + 2 * P.cm;   // 4 records = one 128-byte line
    P.cxy = (long long)P.cx * P.cy;
    if (P.step > 8.0 || (unsigned long long)P.cz * (unsigned long long)P.cxy >= (1ULL << 31)) P.cx = 0;    // marching H unavailable
    {   // face-quad accumulators: orientation a = x, y, z with in-plane axes (b, c) = (y,z), (z,x), (x,y)
        const long long nn[3] = {d.nx, d.ny, d.nz};
        long long tot = 0;
        bool ok = true;
        for (int o = 0; o < 3; ++o) {
            const long long na = nn[o] + 2, nb = nn[(o + 1) % 3] + 1, nc = nn[(o + 2) % 3] + 1;
            if (na * nb * nc >= (1LL << 31)) ok = false;
            P.f_base[o] = tot; P.f_nb[o] = (int)nb; P.f_nc[o] = (int)nc;
            tot += na * nb * nc;
        }
        G->n_faces = ok ? (size_t)tot : 0;
    }
    G->n_cells = P.cx ? (size_t)P.cz * (size_t)P.cxy : 0;
    {   // packed list entries: anchor node offsets in [-128, 895] (anchor = band midpoint, at most 16 samples outside the padded box)
        const int nmax = d.nx > d.ny ? (d.nx > d.nz ? d.nx : d.nz) : (d.ny > d.nz ? d.ny : d.nz);
        // step <= 1: a ray moves at most one cell per sample, which the record-index form of the carry test assumes
        G->march_ok = (P.step <= 1.0) && (16.0 * P.step + 4.0 <= 128.0) && (nmax + 2 + 16.0 * P.step + 4.0 <= 895.0);
    }

    G->n_vox = (size_t)d.nx * d.ny * d.nz;
    G->n_dat = (size_t)Q * K;
    G->n_pad = (size_t)P.pz * P.pxy;
    if (G->n_pad >= (1ULL << 31)) return fail(OAT_ERR_INVALID, "padded grid has more than 2^31 nodes");
    CUDA_TRY(cudaMalloc((void **)&G->d_g, sizeof(double) * (G->n_dat ? G->n_dat : 1)));
    CUDA_TRY(cudaMalloc((void **)&G->d_scal, sizeof(double) * 16));   // [0..7] CG scalars, rest spare
    CUDA_TRY(cudaMalloc((void **)&G->d_counter, sizeof(unsigned long long)));
    CUDA_TRY(cudaMallocHost((void **)&G->h_scal, sizeof(double) * 8));
    CUDA_TRY(cudaEventCreate(&G->ev0));
    CUDA_TRY(cudaEventCreate(&G->ev1));
    if (P.dir) {
        oat_launch_dir_table(P, NB, G->d_dir, 0);
        CUDA_TRY(cudaGetLastError());
        CUDA_TRY(cudaDeviceSynchronize());
    }
    return OAT_OK;
}

int ensure_patches(oat_geometry *G)
{
    if (G->d_patches || G->patch_cap == 0) return OAT_OK;
    long long n = 0;
    const size_t nq = (size_t)(G->dev.Q > 0 ? G->dev.Q : 1);
    if (!G->d_q_count) {
        CUDA_TRY(cudaMalloc((void **)&G->d_q_count, sizeof(int) * nq));
        CUDA_TRY(cudaMalloc((void **)&G->d_q_done, sizeof(int) * nq));
    }
    CUDA_TRY(cudaMemset(G->d_q_count, 0, sizeof(int) * nq));
    G->dev.q_count = G->d_q_count; G->dev.q_done = G->d_q_done;
    cudaError_t e = oat_build_patches(G->dev, G->patch_cap, G->morton_shift, G->d_q_count, &G->d_patches, &n);
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? OAT_ERR_ALLOC : OAT_ERR_CUDA, "patch list generation failed: %s", cudaGetErrorString(e));
    G->dev.patches = G->d_patches;
    G->dev.n_patches = n;
    return OAT_OK;
}

int ensure_xpad(oat_geometry *G)
{
    if (G->d_xpad) return OAT_OK;
    CUDA_TRY(cudaMalloc((void **)&G->d_xpad, sizeof(float) * G->n_pad));
    return OAT_OK;
}

// one traversal of all samples by the generic patch kernel: mode 0 gather, 1 scatter, 2 count
int launch_traversal(oat_geometry *G, int mode, const float *src, float *acc, const float *y, double *g,
                     unsigned long long *counter, cudaStream_t st, bool *launched)
{
    *launched = false;
    int rc = ensure_patches(G); if (rc) return rc;
    if (G->dev.n_patches > 0) { CUDA_TRY(oat_launch_patch(mode, G->dev, src, acc, y, g, counter, st)); *launched = true; }
    return OAT_OK;
}

bool march_h_ok(const oat_geometry *G)
{
    return G->dev.B == 32 && G->n_cells && G->n_cells < G->record_limit && G->dev.dir && G->march_ok;
}

bool march_ht_ok(const oat_geometry *G)
{
    return G->dev.B == 32 && G->n_faces && G->n_faces < G->record_limit && G->dev.dir && G->march_ok;
}

int project_impl(oat_geometry *G, const float *d_x, float *d_y, cudaStream_t st)
{
    const OatDev &P = G->dev;
    G->last_launches = 0;
    if (G->variant_project == 5 && oat_tile_supported(P)) {           // tile-stationary kernel: no patch list, no record array
        CUDA_TRY(cudaMemsetAsync(G->d_g, 0, sizeof(double) * (G->n_dat ? G->n_dat : 1), st));
        CUDA_TRY(cudaEventRecord(G->ev0, st));
        CUDA_TRY(oat_launch_tile_fwd(P, d_x, G->d_g, d_y, G->d_counter, G->d_tile_stats, G->tile_nq, G->tile_tma, st));
        CUDA_TRY(cudaEventRecord(G->ev1, st));
        G->ev_valid = true;
        G->last_launches = 2;
        return OAT_OK;
    }
    const bool march = G->variant_project >= 4 && march_h_ok(G);   // else: B < 32 or a grid the marching kernel cannot index
    int rc = ensure_patches(G); if (rc) return rc;
    if (march) {
        if (!G->d_cells) CUDA_TRY(cudaMalloc((void **)&G->d_cells, sizeof(float4) * 2 * G->n_cells));
        oat_launch_pad_cells(P, d_x, G->d_cells, st); ++G->last_launches;
    } else {
        if ((rc = ensure_xpad(G))) return rc;
        oat_launch_pad(P, d_x, G->d_xpad, st); ++G->last_launches;
    }
    CUDA_TRY(cudaMemsetAsync(G->d_g, 0, sizeof(double) * (G->n_dat ? G->n_dat : 1), st));
    // the kernel that finishes the last patch of a transducer applies 1/t and the time difference itself (step A4)
    if (G->n_dat > 0) CUDA_TRY(cudaMemsetAsync(d_y, 0, sizeof(float) * G->n_dat, st));   // rows without any sample
    if (G->d_q_done) CUDA_TRY(cudaMemsetAsync(G->d_q_done, 0, sizeof(int) * (size_t)(P.Q > 0 ? P.Q : 1), st));
    CUDA_TRY(cudaEventRecord(G->ev0, st));
    bool launched;
    if (march) {
        launched = G->dev.n_patches > 0;
        CUDA_TRY(oat_launch_march(0, G->dev, G->d_cells, nullptr, d_y, nullptr, G->d_g, st));
    } else if ((rc = launch_traversal(G, 0, G->d_xpad, d_y, nullptr, G->d_g, nullptr, st, &launched))) return rc;
    if (launched) ++G->last_launches;
    CUDA_TRY(cudaEventRecord(G->ev1, st));
    G->ev_valid = true;
    CUDA_TRY(cudaGetLastError());
    return OAT_OK;
}

int backproject_impl(oat_geometry *G, const float *d_y, float *d_x, cudaStream_t st)
{
    const OatDev &P = G->dev;
    G->last_launches = 0;
    const bool march = G->variant_backproject >= 4 && march_ht_ok(G);
    int rc = ensure_patches(G); if (rc) return rc;
    if (march) {
        if (!G->d_faces) CUDA_TRY(cudaMalloc((void **)&G->d_faces, sizeof(float4) * G->n_faces));
        CUDA_TRY(cudaMemsetAsync(G->d_faces, 0, sizeof(float4) * G->n_faces, st));
    } else {
        if ((rc = ensure_xpad(G))) return rc;
        CUDA_TRY(cudaMemsetAsync(G->d_xpad, 0, sizeof(float) * G->n_pad, st));
    }
    CUDA_TRY(cudaEventRecord(G->ev0, st));
    bool launched;
    if (march) {
        launched = G->dev.n_patches > 0;
        CUDA_TRY(oat_launch_march(1, G->dev, nullptr, G->d_faces, nullptr, d_y, nullptr, st));
    } else if ((rc = launch_traversal(G, 1, nullptr, G->d_xpad, d_y, nullptr, nullptr, st, &launched))) return rc;
    if (launched) ++G->last_launches;
    CUDA_TRY(cudaEventRecord(G->ev1, st));
    G->ev_valid = true;
    if (march) oat_launch_unface(P, G->d_faces, d_x, st);
    else oat_launch_unpad(P, G->d_xpad, d_x, st);
    ++G->last_launches;
    CUDA_TRY(cudaGetLastError());
    return OAT_OK;
}

int dot_sync(oat_geometry *G, const float *a, const float *b, size_t n, double *out, cudaStream_t st)
{
    CUDA_TRY(cudaMemsetAsync(G->d_scal, 0, sizeof(double), st));
    oat_launch_dot(a, b, (long long)n, G->d_scal, st);
    CUDA_TRY(cudaMemcpyAsync(G->h_scal, G->d_scal, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    *out = G->h_scal[0];
    return OAT_OK;
}

// dot product into slot `i` of the device scalars (asynchronous: the CG loops read it back on the device)
int dot_dev(oat_geometry *G, const float *a, const float *b, size_t n, int i, cudaStream_t st)
{
    CUDA_TRY(cudaMemsetAsync(G->d_scal + i, 0, sizeof(double), st));
    oat_launch_dot(a, b, (long long)n, G->d_scal + i, st);
    return OAT_OK;
}

// pinned curves of a CG run (written by the scalar kernel through UVA), copied to the caller's arrays at the end
struct CgCurves {
    double *a = nullptr, *b = nullptr;
    int n = 0;
    int init(int n_iter, bool want_a, bool want_b)
    {
        n = n_iter + 1;
        if (want_a) CUDA_TRY(cudaMallocHost((void **)&a, sizeof(double) * (size_t)n));
        if (want_b) CUDA_TRY(cudaMallocHost((void **)&b, sizeof(double) * (size_t)n));
        return OAT_OK;
    }
    void finish(double *ha, double *hb)
    {
        if (a && ha) memcpy(ha, a, sizeof(double) * (size_t)n);
        if (b && hb) memcpy(hb, b, sizeof(double) * (size_t)n);
    }
    ~CgCurves() { if (a) cudaFreeHost(a); if (b) cudaFreeHost(b); }
};

// H = H^e D G (Eq. 11) and H^T = G^T D^T H^e† (L168); without taps the EIR is left out
int project_full(oat_geometry *G, const float *d_x, float *d_u, cudaStream_t st)
{
    if (!G->d_he) return project_impl(G, d_x, d_u, st);
    int rc = ensure(&G->d_y4, G->n_dat); if (rc) return rc;
    if ((rc = project_impl(G, d_x, G->d_y4, st))) return rc;
    CUDA_TRY(oat_launch_eir(0, G->d_y4, d_u, G->d_he, G->n_he, G->dev.Q, G->dev.K, st));
    return OAT_OK;
}

int backproject_full(oat_geometry *G, const float *d_u, float *d_x, cudaStream_t st)
{
    if (!G->d_he) return backproject_impl(G, d_u, d_x, st);
    int rc = ensure(&G->d_y4, G->n_dat); if (rc) return rc;
    CUDA_TRY(oat_launch_eir(1, d_u, G->d_y4, G->d_he, G->n_he, G->dev.Q, G->dev.K, st));
    return backproject_impl(G, G->d_y4, d_x, st);
}

int check_handle(const oat_geometry *g)
{
    if (!g) return fail(OAT_ERR_INVALID, "geometry handle is NULL");
    cudaError_t e = cudaSetDevice(g->device);
    if (e != cudaSuccess) return fail(OAT_ERR_CUDA, "cudaSetDevice(%d) failed: %s", g->device, cudaGetErrorString(e));
    return OAT_OK;
}

}  // namespace

extern "C" {

int oat_geometry_create(const oat_geometry_desc *desc, int device, oat_geometry **out)
{
    if (!desc || !out) return fail(OAT_ERR_INVALID, "desc and out must not be NULL");
    if (desc->nx < 1 || desc->ny < 1 || desc->nz < 1) return fail(OAT_ERR_INVALID, "grid sizes must be >= 1");
    if ((long long)desc->nx * desc->ny * desc->nz > (1LL << 40)) return fail(OAT_ERR_INVALID, "grid too large");
    if (desc->n_trans < 0 || desc->nt < 1) return fail(OAT_ERR_INVALID, "n_trans must be >= 0 and nt >= 1");
    if (!(desc->spacing > 0) || !(desc->c > 0) || !(desc->dt > 0) || !(desc->t0 >= 0))
        return fail(OAT_ERR_INVALID, "spacing, c, dt must be > 0 and t0 >= 0");
    if (!isfinite(desc->spacing) || !isfinite(desc->c) || !isfinite(desc->dt) || !isfinite(desc->t0))
        return fail(OAT_ERR_INVALID, "non-finite scalar in descriptor");
    if (desc->surf_step < 0 || !isfinite(desc->surf_step)) return fail(OAT_ERR_INVALID, "surf_step must be >= 0");
    if (desc->kband < 0 || desc->kband > 32) return fail(OAT_ERR_INVALID, "kband must be in 0..32");
    if (!isfinite(desc->gain)) return fail(OAT_ERR_INVALID, "gain must be finite");
    if (desc->n_trans > 0 && !desc->trans_xyz) return fail(OAT_ERR_INVALID, "trans_xyz is NULL");
    for (int a = 0; a < 3; ++a)
        if (!isfinite(desc->origin[a])) return fail(OAT_ERR_INVALID, "origin must be finite");
    for (long long i = 0; i < 3LL * desc->n_trans; ++i)
        if (!isfinite(desc->trans_xyz[i])) return fail(OAT_ERR_INVALID, "transducer %lld has a non-finite coordinate", i / 3);
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev <= 0)
        return fail(OAT_ERR_CUDA, "no CUDA device (%s); liboat has no CPU fallback", e != cudaSuccess ? cudaGetErrorString(e) : "count = 0");
    if (device < 0 || device >= ndev) return fail(OAT_ERR_INVALID, "device %d out of range (0..%d)", device, ndev - 1);
    CUDA_TRY(cudaSetDevice(device));

    oat_geometry *G = new (std::nothrow) oat_geometry();
    if (!G) return fail(OAT_ERR_ALLOC, "out of host memory");
    G->desc = *desc;
    G->device = device;
    std::vector<double> tr_copy;
    try {
        tr_copy.assign(desc->trans_xyz, desc->trans_xyz + 3 * (size_t)desc->n_trans);
    } catch (...) { delete G; return fail(OAT_ERR_ALLOC, "out of host memory"); }
    G->desc.trans_xyz = tr_copy.data();
    int rc;
    try { rc = build_geometry(G); }
    catch (const std::bad_alloc &) { rc = fail(OAT_ERR_ALLOC, "out of host memory while building tables"); }
    G->desc.trans_xyz = nullptr;                           // the copy lives on the device (frames) only
    if (rc) { free_all(G); return rc; }
    *out = G;
    return OAT_OK;
}

void oat_geometry_destroy(oat_geometry *geom)
{
    if (!geom) return;
    cudaSetDevice(geom->device);
    free_all(geom);
}

int64_t oat_num_voxels(const oat_geometry *g) { return g ? (int64_t)g->n_vox : -1; }
int64_t oat_num_samples(const oat_geometry *g) { return g ? (int64_t)g->n_dat : -1; }

int64_t oat_num_surface_samples(oat_geometry *g)
{
    if (check_handle(g)) return -1;
    if (g->n_surface_samples >= 0) return g->n_surface_samples;
    if (cudaMemset(g->d_counter, 0, sizeof(unsigned long long)) != cudaSuccess) return -1;
    bool launched;
    if (launch_traversal(g, 2, nullptr, nullptr, nullptr, nullptr, g->d_counter, 0, &launched)) return -1;
    unsigned long long v = 0;
    if (cudaMemcpy(&v, g->d_counter, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) {
        fail(OAT_ERR_CUDA, "sample count kernel failed: %s", cudaGetErrorString(cudaGetLastError()));
        return -1;
    }
    g->n_surface_samples = (long long)v;
    return g->n_surface_samples;
}

int oat_project(oat_geometry *g, const float *d_x, float *d_y, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || (!d_y && g->n_dat)) return fail(OAT_ERR_INVALID, "d_x / d_y must not be NULL");
    return project_impl(g, d_x, d_y, (cudaStream_t)stream);
}

int oat_backproject(oat_geometry *g, const float *d_y, float *d_x, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || (!d_y && g->n_dat)) return fail(OAT_ERR_INVALID, "d_x / d_y must not be NULL");
    return backproject_impl(g, d_y, d_x, (cudaStream_t)stream);
}

int oat_adjoint_check(oat_geometry *g, const float *d_x, const float *d_y, double *lhs, double *rhs, double *rel, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || !d_y || !lhs || !rhs || !rel) return fail(OAT_ERR_INVALID, "NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = ensure(&g->d_y2, g->n_dat))) return rc;
    if ((rc = ensure(&g->d_x2, g->n_vox))) return rc;
    if ((rc = project_impl(g, d_x, g->d_y2, st))) return rc;
    if ((rc = dot_sync(g, g->d_y2, d_y, g->n_dat, lhs, st))) return rc;
    if ((rc = backproject_impl(g, d_y, g->d_x2, st))) return rc;
    if ((rc = dot_sync(g, d_x, g->d_x2, g->n_vox, rhs, st))) return rc;
    const double m = fmax(fabs(*lhs), fabs(*rhs));
    *rel = m > 0 ? fabs(*lhs - *rhs) / m : 0.0;
    return OAT_OK;
}

int oat_project_host(oat_geometry *g, const float *h_x, float *h_y)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!h_x || (!h_y && g->n_dat)) return fail(OAT_ERR_INVALID, "h_x / h_y must not be NULL");
    if ((rc = ensure(&g->d_y2, g->n_dat))) return rc;
    if ((rc = ensure(&g->d_x2, g->n_vox))) return rc;
    CUDA_TRY(cudaMemcpyAsync(g->d_x2, h_x, sizeof(float) * g->n_vox, cudaMemcpyHostToDevice, 0));
    if ((rc = project_impl(g, g->d_x2, g->d_y2, 0))) return rc;
    CUDA_TRY(cudaMemcpyAsync(h_y, g->d_y2, sizeof(float) * g->n_dat, cudaMemcpyDeviceToHost, 0));
    CUDA_TRY(cudaStreamSynchronize(0));
    return OAT_OK;
}

int oat_backproject_host(oat_geometry *g, const float *h_y, float *h_x)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!h_x || (!h_y && g->n_dat)) return fail(OAT_ERR_INVALID, "h_x / h_y must not be NULL");
    if ((rc = ensure(&g->d_y2, g->n_dat))) return rc;
    if ((rc = ensure(&g->d_x2, g->n_vox))) return rc;
    CUDA_TRY(cudaMemcpyAsync(g->d_y2, h_y, sizeof(float) * g->n_dat, cudaMemcpyHostToDevice, 0));
    if ((rc = backproject_impl(g, g->d_y2, g->d_x2, 0))) return rc;
    CUDA_TRY(cudaMemcpyAsync(h_x, g->d_x2, sizeof(float) * g->n_vox, cudaMemcpyDeviceToHost, 0));
    CUDA_TRY(cudaStreamSynchronize(0));
    return OAT_OK;
}

// Row C1: CGLS (reading G15).  r = y - Hx; s = H^T r; p = s; loop { q = Hp; alpha = |s|^2/|q|^2;
// x += alpha p; r -= alpha q; s = H^T r; beta = |s|^2_new/|s|^2_old; p = s + beta p }
int oat_cgls(oat_geometry *g, const float *d_y, float *d_x, int n_iter, double *h_res, double *h_grad, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_y || !d_x || n_iter < 0) return fail(OAT_ERR_INVALID, "bad argument to oat_cgls");
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = ensure(&g->d_y2, g->n_dat))) return rc;     // r
    if ((rc = ensure(&g->d_y3, g->n_dat))) return rc;     // q
    if ((rc = ensure(&g->d_x3, g->n_vox))) return rc;     // s
    if ((rc = ensure(&g->d_x4, g->n_vox))) return rc;     // p
    float *r = g->d_y2, *qv = g->d_y3, *s = g->d_x3, *p = g->d_x4;
    // scalars stay on the device (slots: oat_kernels.cu, oat_cg_scalar_kernel); ONE synchronisation, at the end
    CgCurves cv;
    if ((rc = cv.init(n_iter, h_res != nullptr, h_grad != nullptr))) return rc;
    double *sc = g->d_scal;
    CUDA_TRY(cudaMemsetAsync(d_x, 0, sizeof(float) * g->n_vox, st));
    CUDA_TRY(cudaMemcpyAsync(r, d_y, sizeof(float) * g->n_dat, cudaMemcpyDeviceToDevice, st));
    if ((rc = backproject_impl(g, r, s, st))) return rc;
    CUDA_TRY(cudaMemcpyAsync(p, s, sizeof(float) * g->n_vox, cudaMemcpyDeviceToDevice, st));
    if ((rc = dot_dev(g, s, s, g->n_vox, 0, st))) return rc;               // gamma
    if ((rc = dot_dev(g, d_y, d_y, g->n_dat, 6, st))) return rc;           // |y|^2
    oat_launch_cg_scalar(sc, 0, 0, 0.0, cv.a, cv.b, st);
    for (int it = 0; it < n_iter; ++it) {
        if ((rc = project_impl(g, p, qv, st))) return rc;
        if ((rc = dot_dev(g, qv, qv, g->n_dat, 1, st))) return rc;
        oat_launch_cg_scalar(sc, 1, it, 0.0, nullptr, nullptr, st);         // alpha = gamma / |q|^2 (flag 0: leave everything as it is)
        oat_launch_axpy_dev(sc, 3, 7, 1.f, p, d_x, (long long)g->n_vox, st);
        oat_launch_axpy_dev(sc, 3, 7, -1.f, qv, r, (long long)g->n_dat, st);
        if ((rc = backproject_impl(g, r, s, st))) return rc;
        if ((rc = dot_dev(g, s, s, g->n_vox, 2, st))) return rc;
        oat_launch_cg_scalar(sc, 2, it, 0.0, nullptr, nullptr, st);         // beta, gamma
        oat_launch_xpay_dev(s, sc, 4, 7, p, (long long)g->n_vox, st);
        if (h_res && (rc = dot_dev(g, r, r, g->n_dat, 5, st))) return rc;
        oat_launch_cg_scalar(sc, 3, it, 0.0, cv.a, cv.b, st);
    }
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(st));
    cv.finish(h_res, h_grad);
    return OAT_OK;
}

int oat_eir_set(oat_geometry *g, const float *h_he, int32_t len)
{
    int rc = check_handle(g); if (rc) return rc;
    if (len < 0 || (len > 0 && !h_he)) return fail(OAT_ERR_INVALID, "bad EIR taps");
    if (len > 16384) return fail(OAT_ERR_INVALID, "EIR longer than 16384 taps");
    for (int i = 0; i < len; ++i) if (!isfinite(h_he[i])) return fail(OAT_ERR_INVALID, "EIR tap %d is not finite", i);
    CUDA_TRY(cudaDeviceSynchronize());                    // the old taps may still be in use
    cudaFree(g->d_he); g->d_he = nullptr; g->n_he = 0;
    if (len == 0) return OAT_OK;
    CUDA_TRY(cudaMalloc((void **)&g->d_he, sizeof(float) * (size_t)len));
    CUDA_TRY(cudaMemcpy(g->d_he, h_he, sizeof(float) * (size_t)len, cudaMemcpyHostToDevice));
    g->n_he = len;
    return OAT_OK;
}

int oat_eir_apply(oat_geometry *g, const float *d_in, float *d_out, int adjoint, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if ((!d_in || !d_out) && g->n_dat) return fail(OAT_ERR_INVALID, "d_in / d_out must not be NULL");
    if (d_in == d_out && g->n_dat) return fail(OAT_ERR_INVALID, "oat_eir_apply cannot run in place");
    if (!g->d_he) return fail(OAT_ERR_INVALID, "no EIR set (oat_eir_set)");
    CUDA_TRY(oat_launch_eir(adjoint ? 1 : 0, d_in, d_out, g->d_he, g->n_he, g->dev.Q, g->dev.K, (cudaStream_t)stream));
    return OAT_OK;
}

int oat_penalty_apply(oat_geometry *g, const float *d_x, float *d_lx, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || !d_lx || d_x == d_lx) return fail(OAT_ERR_INVALID, "d_x / d_lx must be distinct non-NULL buffers");
    oat_launch_penalty(g->dev, d_x, d_lx, 1.f, 0.f, (cudaStream_t)stream);
    CUDA_TRY(cudaGetLastError());
    return OAT_OK;
}

int oat_penalty_value(oat_geometry *g, const float *d_x, double *value, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || !value) return fail(OAT_ERR_INVALID, "NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = ensure(&g->d_x2, g->n_vox))) return rc;
    oat_launch_penalty(g->dev, d_x, g->d_x2, 1.f, 0.f, st);
    return dot_sync(g, d_x, g->d_x2, g->n_vox, value, st);   // R(x) = x^T L x
}

int oat_project_eir(oat_geometry *g, const float *d_x, float *d_u, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || (!d_u && g->n_dat)) return fail(OAT_ERR_INVALID, "d_x / d_u must not be NULL");
    return project_full(g, d_x, d_u, (cudaStream_t)stream);
}

int oat_backproject_eir(oat_geometry *g, const float *d_u, float *d_x, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || (!d_u && g->n_dat)) return fail(OAT_ERR_INVALID, "d_x / d_u must not be NULL");
    return backproject_full(g, d_u, d_x, (cudaStream_t)stream);
}

// Rows NEXT-1 / NEXT-3 (reading G22): linear CG on (H^T H + mu L) x = H^T u from x = 0.  sph = false: H = H^e D G, data =
// Q*K floats (Eq. 29); sph = true: H = H_sph, data = Q*nf complex numbers handled as 2*Q*nf floats -- the real inner
// product of the interleaved (re, im) pairs is Re<.,.> of C^{QL} (Eq. 30, reading G29).
static int pls_cg_impl(oat_geometry *g, const float *d_u, float *d_x, int n_iter, double mu, double *h_obj, double *h_grad,
                       cudaStream_t st, bool sph)
{
    int rc;
    const size_t n_dat = sph ? 2 * (size_t)g->sph_nf * (size_t)g->dev.Q : g->n_dat;
    float **pd = sph ? &g->d_sd : &g->d_y2, **pq = sph ? &g->d_sq : &g->d_y3;
    if ((rc = ensure(pd, n_dat))) return rc;                // d = u - H x
    if ((rc = ensure(pq, n_dat))) return rc;                // q = H p
    if ((rc = ensure(&g->d_x2, g->n_vox))) return rc;     // w = (H^T H + mu L) p, later L x
    if ((rc = ensure(&g->d_x3, g->n_vox))) return rc;     // r
    if ((rc = ensure(&g->d_x4, g->n_vox))) return rc;     // p
    float *d = *pd, *q = *pq, *w = g->d_x2, *r = g->d_x3, *p = g->d_x4;
    auto fwd = [&](const float *x, float *u) -> int {
        if (!sph) return project_full(g, x, u, st);
        CUDA_TRY(cudaMemsetAsync(u, 0, sizeof(float) * n_dat, st));
        CUDA_TRY(oat_launch_sph_fwd(g->dev, g->sph_nf, g->sph_f0, g->sph_df, g->desc.spacing, g->desc.c, g->sph_aperture, g->sph_m, x, g->d_p0, u, st));
        return OAT_OK;
    };
    auto bwd = [&](const float *u, float *x) -> int {
        if (!sph) return backproject_full(g, u, x, st);
        oat_launch_sph_bwd(g->dev, g->sph_nf, g->sph_f0, g->sph_df, g->desc.spacing, g->desc.c, g->sph_aperture, g->sph_m,
                           reinterpret_cast<const float2 *>(u), g->d_p0, g->d_sv, x, st);
        CUDA_TRY(cudaGetLastError());                      // a bad launch surfaces here, not after the whole loop has been enqueued
        return OAT_OK;
    };
    CgCurves cv;
    if ((rc = cv.init(n_iter, h_obj != nullptr, h_grad != nullptr))) return rc;
    double *sc = g->d_scal;
    CUDA_TRY(cudaMemsetAsync(d_x, 0, sizeof(float) * g->n_vox, st));
    CUDA_TRY(cudaMemcpyAsync(d, d_u, sizeof(float) * n_dat, cudaMemcpyDeviceToDevice, st));
    if ((rc = bwd(d_u, r))) return rc;
    CUDA_TRY(cudaMemcpyAsync(p, r, sizeof(float) * g->n_vox, cudaMemcpyDeviceToDevice, st));
    if ((rc = dot_dev(g, r, r, g->n_vox, 0, st))) return rc;               // |r|^2
    if ((rc = dot_dev(g, d, d, n_dat, 5, st))) return rc;                  // |u|^2
    oat_launch_cg_scalar(sc, 4, 0, mu, cv.a, cv.b, st);
    for (int it = 0; it < n_iter; ++it) {
        if ((rc = fwd(p, q))) return rc;
        if ((rc = bwd(q, w))) return rc;
        if (mu > 0) oat_launch_penalty(g->dev, p, w, (float)mu, 1.f, st);          // w += mu L p
        if ((rc = dot_dev(g, p, w, g->n_vox, 1, st))) return rc;
        oat_launch_cg_scalar(sc, 1, it, mu, nullptr, nullptr, st);         // alpha = |r|^2 / <p, w> (flag 0: a degenerate step changes nothing)
        oat_launch_axpy_dev(sc, 3, 7, 1.f, p, d_x, (long long)g->n_vox, st);
        oat_launch_axpy_dev(sc, 3, 7, -1.f, q, d, (long long)n_dat, st);
        oat_launch_axpy_dev(sc, 3, 7, -1.f, w, r, (long long)g->n_vox, st);
        if ((rc = dot_dev(g, r, r, g->n_vox, 2, st))) return rc;
        oat_launch_cg_scalar(sc, 2, it, mu, nullptr, nullptr, st);         // beta, |r|^2
        oat_launch_xpay_dev(r, sc, 4, 7, p, (long long)g->n_vox, st);
        if (h_obj) {
            if ((rc = dot_dev(g, d, d, n_dat, 5, st))) return rc;
            CUDA_TRY(cudaMemsetAsync(sc + 6, 0, sizeof(double), st));
            if (mu > 0) {
                oat_launch_penalty(g->dev, d_x, w, 1.f, 0.f, st);
                oat_launch_dot(d_x, w, (long long)g->n_vox, sc + 6, st);
            }
        }
        oat_launch_cg_scalar(sc, 5, it, mu, cv.a, cv.b, st);
    }
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(st));
    cv.finish(h_obj, h_grad);
    return OAT_OK;
}

int oat_pls_cg(oat_geometry *g, const float *d_u, float *d_x, int n_iter, double mu, double *h_obj, double *h_grad, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_u || !d_x || n_iter < 0 || !(mu >= 0) || !isfinite(mu)) return fail(OAT_ERR_INVALID, "bad argument to oat_pls_cg");
    return pls_cg_impl(g, d_u, d_x, n_iter, mu, h_obj, h_grad, (cudaStream_t)stream, false);
}

int oat_sph_pls_cg(oat_geometry *g, const float *d_u, float *d_x, int n_iter, double mu, double *h_obj, double *h_grad, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!g->sph_nf) return fail(OAT_ERR_INVALID, "no frequency grid set (oat_sph_set)");
    if (!d_u || !d_x || n_iter < 0 || !(mu >= 0) || !isfinite(mu)) return fail(OAT_ERR_INVALID, "bad argument to oat_sph_pls_cg");
    return pls_cg_impl(g, d_u, d_x, n_iter, mu, h_obj, h_grad, (cudaStream_t)stream, true);
}

int oat_sph_set(oat_geometry *g, int32_t nf, double f0, double df, const float *h_he)
{
    int rc = check_handle(g); if (rc) return rc;
    if (nf < 0 || nf > (1 << 20) || !(f0 >= 0) || !(df >= 0) || !isfinite(f0) || !isfinite(df))
        return fail(OAT_ERR_INVALID, "bad frequency grid (nf >= 0, f0 >= 0, df >= 0)");
    CUDA_TRY(cudaDeviceSynchronize());
    cudaFree(g->d_p0); cudaFree(g->d_sv); cudaFree(g->d_sd); cudaFree(g->d_sq);
    g->d_p0 = nullptr; g->d_sv = nullptr; g->d_sd = nullptr; g->d_sq = nullptr; g->sph_nf = 0;
    if (nf == 0) return OAT_OK;
    // Eq. (19) L153 in fp64 (reading G27): p~0(f) = -j (4 pi kappa c^3 / f) [ (ds/2c) cos(pi f ds/c) - sin(pi f ds/c)/(2 pi f) ] h~e(f), p~0(0) = 0
    std::vector<float2> p0((size_t)nf);
    const double ds = g->desc.spacing, c = g->desc.c;
    for (int l = 0; l < nf; ++l) {
        const double f = f0 + l * df;
        double im = 0.0;
        if (f != 0.0) {
            const double a = kPi * f * ds / c;
            im = -(4.0 * kPi * g->kappa * c * c * c / f) * ((ds / (2.0 * c)) * cos(a) - sin(a) / (2.0 * kPi * f));
        }
        double re = 0.0;
        if (h_he) {                                        // (j im) (hr + j hi) = -im hi + j im hr
            const double hr = h_he[2 * l], hi = h_he[2 * l + 1];
            if (!isfinite(hr) || !isfinite(hi)) return fail(OAT_ERR_INVALID, "EIR spectrum sample %d is not finite", l);
            re = -im * hi; im = im * hr;
        }
        p0[l] = make_float2((float)re, (float)im);
    }
    CUDA_TRY(cudaMalloc((void **)&g->d_p0, sizeof(float2) * (size_t)nf));
    CUDA_TRY(cudaMemcpy(g->d_p0, p0.data(), sizeof(float2) * (size_t)nf, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMalloc((void **)&g->d_sv, sizeof(float2) * (size_t)nf * (size_t)(g->dev.Q > 0 ? g->dev.Q : 1)));
    g->sph_nf = nf; g->sph_f0 = f0; g->sph_df = df;
    return OAT_OK;
}

int oat_sph_set_aperture(oat_geometry *g, double side, int32_t m)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!(side >= 0) || !isfinite(side) || m < 1 || m > 64) return fail(OAT_ERR_INVALID, "bad aperture (side >= 0, 1 <= m <= 64)");
    CUDA_TRY(cudaDeviceSynchronize());
    g->sph_aperture = side; g->sph_m = m;
    return OAT_OK;
}

int oat_sph_project(oat_geometry *g, const float *d_x, float *d_u, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!g->sph_nf) return fail(OAT_ERR_INVALID, "no frequency grid set (oat_sph_set)");
    if (!d_x || (!d_u && g->dev.Q)) return fail(OAT_ERR_INVALID, "d_x / d_u must not be NULL");
    cudaStream_t st = (cudaStream_t)stream;
    if (g->dev.Q > 0) CUDA_TRY(cudaMemsetAsync(d_u, 0, sizeof(float2) * (size_t)g->sph_nf * (size_t)g->dev.Q, st));
    CUDA_TRY(oat_launch_sph_fwd(g->dev, g->sph_nf, g->sph_f0, g->sph_df, g->desc.spacing, g->desc.c, g->sph_aperture, g->sph_m, d_x, g->d_p0, d_u, st));
    return OAT_OK;
}

int oat_sph_backproject(oat_geometry *g, const float *d_u, float *d_x, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!g->sph_nf) return fail(OAT_ERR_INVALID, "no frequency grid set (oat_sph_set)");
    if (!d_x || (!d_u && g->dev.Q)) return fail(OAT_ERR_INVALID, "d_x / d_u must not be NULL");
    oat_launch_sph_bwd(g->dev, g->sph_nf, g->sph_f0, g->sph_df, g->desc.spacing, g->desc.c, g->sph_aperture, g->sph_m,
                       reinterpret_cast<const float2 *>(d_u), g->d_p0, g->d_sv, d_x, (cudaStream_t)stream);
    CUDA_TRY(cudaGetLastError());
    return OAT_OK;
}

int oat_fbp(oat_geometry *g, const float *d_p, const float *d_w, float *d_x, void *stream)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!d_x || ((!d_p || !d_w) && g->n_dat)) return fail(OAT_ERR_INVALID, "d_p / d_w / d_x must not be NULL");
    if (g->dev.K < 2) { CUDA_TRY(cudaMemsetAsync(d_x, 0, sizeof(float) * g->n_vox, (cudaStream_t)stream)); return OAT_OK; }
    oat_launch_fbp(g->dev, d_p, d_w, d_x, (cudaStream_t)stream);
    CUDA_TRY(cudaGetLastError());
    return OAT_OK;
}

int oat_fbp_weights(const oat_geometry *g, const double *h_areas, float *h_w)
{
    if (!g) return fail(OAT_ERR_INVALID, "geometry handle is NULL");
    if ((!h_areas || !h_w) && g->dev.Q) return fail(OAT_ERR_INVALID, "h_areas / h_w must not be NULL");
    const double c = g->desc.c, k = 4.0 * kPi * kPi * g->kappa * c * c * c * g->desc.dt;
    for (int q = 0; q < g->dev.Q; ++q) h_w[q] = (float)(-h_areas[q] / (k * g->h_rq[(size_t)q]));
    return OAT_OK;
}

int oat_set_variant(oat_geometry *g, const char *key, int variant)
{
    if (!g || !key) return fail(OAT_ERR_INVALID, "NULL argument");
    if (!strcmp(key, "project")) { if (variant != 0 && variant != 4 && variant != 5) return fail(OAT_ERR_INVALID, "unknown project variant %d (0 generic, 4 marching, 5 tile-stationary)", variant); g->variant_project = variant; return OAT_OK; }
    if (!strcmp(key, "tile_nq")) { if (variant < 1) return fail(OAT_ERR_INVALID, "tile_nq must be >= 1"); g->tile_nq = variant; return OAT_OK; }
    if (!strcmp(key, "tile_tma")) { g->tile_tma = variant ? 1 : 0; return OAT_OK; }
    if (!strcmp(key, "tile_stats")) {
        if (variant && !g->d_tile_stats) {
            CUDA_TRY(cudaMalloc((void **)&g->d_tile_stats, sizeof(unsigned long long) * 8));
            CUDA_TRY(cudaMemset(g->d_tile_stats, 0, sizeof(unsigned long long) * 8));
        } else if (!variant && g->d_tile_stats) { CUDA_TRY(cudaDeviceSynchronize()); cudaFree(g->d_tile_stats); g->d_tile_stats = nullptr; }
        return OAT_OK;
    }
    if (!strcmp(key, "backproject")) {
        // variant 5 (tile-stationary H^T, int32 fixed-point accumulators in shared memory) was measured in round 2 and removed:
        // 2.05x slower and 8e-5 .. 5.7e-4 from the oracle, with no overflow guard.  A handle cannot be switched onto it.
        if (variant == 5) return fail(OAT_ERR_INVALID, "backproject variant 5 (tile-stationary H^T) is not part of the library: it missed the 1e-4 tolerance (profiles/r2_tile_bwd.md)");
        if (variant != 0 && variant != 4) return fail(OAT_ERR_INVALID, "unknown backproject variant %d (0 generic, 4 marching)", variant);
        g->variant_backproject = variant; return OAT_OK;
    }
    if (!strcmp(key, "morton_shift")) {
        if (variant < 0 || variant > 10) return fail(OAT_ERR_INVALID, "morton_shift out of range");
        if (g->morton_shift != variant) { cudaFree(g->d_patches); g->d_patches = nullptr; g->dev.patches = nullptr; g->dev.n_patches = 0; }
        g->morton_shift = variant; return OAT_OK;
    }
    if (!strcmp(key, "record_limit_log2")) {               // tests: pretend the 32-bit record index is narrower
        if (variant < 1 || variant > 31) return fail(OAT_ERR_INVALID, "record_limit_log2 out of range");
        g->record_limit = (size_t)1 << variant; return OAT_OK;
    }
    return fail(OAT_ERR_INVALID, "unknown variant key '%s'", key);
}

int oat_uses_marching(const oat_geometry *g, int backproject)
{
    if (!g) return -1;
    return backproject ? (g->variant_backproject == 4 && march_ht_ok(g)) : (g->variant_project == 4 && march_h_ok(g));
}

int oat_tile_stats(oat_geometry *g, unsigned long long *h_out, int reset)
{
    int rc = check_handle(g); if (rc) return rc;
    if (!h_out || !g->d_tile_stats) return fail(OAT_ERR_INVALID, "tile statistics are off (oat_set_variant(g, \"tile_stats\", 1))");
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpy(h_out, g->d_tile_stats, sizeof(unsigned long long) * 8, cudaMemcpyDeviceToHost));
    if (reset) CUDA_TRY(cudaMemset(g->d_tile_stats, 0, sizeof(unsigned long long) * 8));
    return OAT_OK;
}

int oat_last_launch_count(const oat_geometry *g) { return g ? g->last_launches : -1; }

float oat_last_kernel_ms(oat_geometry *g)
{
    if (check_handle(g) || !g->ev_valid) return -1.f;
    if (cudaEventSynchronize(g->ev1) != cudaSuccess) return -1.f;
    float ms = -1.f;
    if (cudaEventElapsedTime(&ms, g->ev0, g->ev1) != cudaSuccess) return -1.f;
    return ms;
}

const char *oat_last_error(void) { return g_err; }
const char *oat_version(void) { return "oat-b200 0.1 (OAT-DISC v1; sm_100a)"; }

}  // extern "C"
