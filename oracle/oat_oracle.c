/*
 * oat_oracle.c -- fp64 CPU ORACLE for the matched projector pair H = D.G and
 * H^T = G^T.D^T of the interpolation-based D-D imaging model of 3-D OAT
 * (arxiv/paper_1304_2017: Eq. (2)-(3) L59-63; Eq. (10)-(13) L110-125;
 * Eq. (22)-(23) L172-177; Appendix Eq. (35)-(39) L346-366; Alg. 4;
 * Alg. 6).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check
 * of __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it.  It shares no code, header, table or constant with
 * the CUDA library (paper_1304_2017_b200/csrc); neither includes the other.
 *
 * It is the discretisation "OAT-DISC v1"
 * written out step by step in the paper's order and notation, in double
 * precision, with no blocking, fusion or reordering:
 *
 *     for every transducer q            (Eq. 5: data index m = q*K + k)
 *       for every time sample k         (t_k = t0 + k dt, rho_k = c t_k)
 *         for every ring i              (theta_i = i dtheta,  Eq. 38)
 *           for every azimuth j         (phi_j = j dphi,      Eq. 38)
 *             sample, interpolate trilinearly (Eq. 10), accumulate
 *
 * The only deviation from a literal whole-sphere loop is the S9 cull: rings
 * that provably miss the ball circumscribing the zero-padded node box are not
 * visited (this is the paper's own theta'_max, Alg. 4) and samples outside
 * the padded box are skipped; both discard only terms that are exactly zero.
 *
 * Pins (tests/test_oracle_pins.py): closed-form spherical means of a uniform
 * ball and of a Gaussian (P1, P2), quadrature weight sum 4 pi (P3), adjoint
 * identity to 1e-12 (P4), brute-force dense matrix from the hat-function
 * definition on tiny grids (P5), N-wave of a ball (P6), D on quadratics and
 * D^T against the explicit transpose (P7), structural cases (P8).
 * Agreement with the AUTHORS' implementation is "parity unpinned": the paper
 * prints no value of g, p or alpha'.
 *
 * OpenMP is used only to run independent transducers on several cores; the
 * arithmetic per transducer is the plain loop above.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define OAT_REF_OK 0
#define OAT_REF_ERR_INVALID (-1)
#define OAT_REF_ERR_ALLOC (-2)

/* Problem statement of the paper (L203; point-like transducers L114). */
typedef struct {
    int32_t nx, ny, nz;        /* nodes per axis */
    double spacing;            /* Delta_s */
    double origin[3];          /* node (0,0,0) = (x_min, y_min, z_min) */
    int32_t n_trans;           /* Q */
    const double *trans_xyz;   /* Q x 3, host */
    double c, t0, dt;          /* c_0, t_min, Delta_t */
    int32_t nt;                /* K */
    double surf_step;          /* h (0 => spacing, Eq. 37) */
    int32_t kband;             /* B (0 => 32; 1 = per-sample angular step) */
    double gain;               /* kappa = beta/(4 pi C_p) (0 => 1) */
    int32_t literal;           /* reading G2 switch: 1 => N_j = floor(2 pi / dphi),
                                  patch weight h^2 exactly as printed in Eq. (37)-(38);
                                  for comparison only, never the parity target */
    int32_t n_threads;         /* 0 => OpenMP default */
} oat_ref_desc;

typedef struct {
    double h, kappa;
    int B;
    double C[3];               /* grid centre (S0) */
    double r_pad;              /* radius of the ball around C containing the padded box */
} ref_consts;

static int ref_setup(const oat_ref_desc *d, ref_consts *k)
{
    if (!d || d->nx <= 0 || d->ny <= 0 || d->nz <= 0 || d->n_trans < 0 || d->nt <= 0) return OAT_REF_ERR_INVALID;
    if (!(d->spacing > 0) || !(d->c > 0) || !(d->dt > 0) || !(d->t0 >= 0)) return OAT_REF_ERR_INVALID;
    if (d->n_trans > 0 && !d->trans_xyz) return OAT_REF_ERR_INVALID;
    if (d->surf_step < 0 || d->kband < 0) return OAT_REF_ERR_INVALID;
    k->h = d->surf_step > 0 ? d->surf_step : d->spacing;
    k->B = d->kband > 0 ? d->kband : 32;
    k->kappa = d->gain != 0 ? d->gain : 1.0;
    const int n[3] = {d->nx, d->ny, d->nz};
    double r2 = 0;
    for (int a = 0; a < 3; ++a) {
        k->C[a] = d->origin[a] + d->spacing * 0.5 * (n[a] - 1);       /* S0 */
        double half = d->spacing * (0.5 * (n[a] - 1) + 1.0);           /* padded by one node */
        r2 += half * half;
    }
    k->r_pad = sqrt(r2);
    return OAT_REF_OK;
}

/* S1: local frame at the transducer; z^tr points to the grid centre (Appendix). */
static int ref_frame(const ref_consts *k, const double *rq, double ex[3], double ey[3], double ez[3], double *L)
{
    double v[3] = {k->C[0] - rq[0], k->C[1] - rq[1], k->C[2] - rq[2]};
    double len = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    if (!(len > 0)) return OAT_REF_ERR_INVALID;
    for (int a = 0; a < 3; ++a) ez[a] = v[a] / len;
    double ax = ez[1], ay = -ez[0];                /* a = e_z x z^ = (ez.y, -ez.x, 0) */
    double an = sqrt(ax * ax + ay * ay);
    if (an < 1e-12) { ey[0] = 0; ey[1] = 1; ey[2] = 0; }
    else { ey[0] = ax / an; ey[1] = ay / an; ey[2] = 0; }
    ex[0] = ey[1] * ez[2] - ey[2] * ez[1];         /* e_x = e_y x e_z */
    ex[1] = ey[2] * ez[0] - ey[0] * ez[2];
    ex[2] = ey[0] * ez[1] - ey[1] * ez[0];
    *L = len;
    return OAT_REF_OK;
}

/* S9: largest polar angle at which the shell of radius rho can meet the ball of
 * radius r_pad around the grid centre (paper's theta'_max, Alg. 4).
 * Returns a negative value when the shell misses the ball altogether. */
static double ref_theta_max(double L, double rho, double R)
{
    if (rho >= L + R) return -1.0;                  /* shell passes beyond the ball */
    if (rho <= L - R) return -1.0;                  /* shell does not reach the ball */
    if (rho <= R - L) return M_PI;                  /* shell entirely inside the ball */
    /* a shell point at polar angle theta is at distance^2 rho^2 + L^2 - 2 rho L cos(theta) from C */
    double cm = (L * L + rho * rho - R * R) / (2.0 * rho * L);
    if (cm >= 1.0) return -1.0;
    if (cm <= -1.0) return M_PI;
    return acos(cm);
}

/*
 * One traversal of the quadrature of (q, k).  mode 0: gather (S4-S5) and
 * return sum_ij omega * A~(r);  mode 1: scatter (S8) `coef * omega * w` into x;
 * mode 2: count in-box samples.  The three modes share the loop so that G and
 * G^T visit exactly the same samples with exactly the same weights (Eq. 12 vs
 * Eq. 23; Alg. 4 vs Alg. 6 have the same double loop).
 */
static double ref_shell(const oat_ref_desc *d, const ref_consts *kc,
                        const double *rq, const double ex[3], const double ey[3], const double ez[3], double L,
                        int k, int mode, const double *x, double *xs, double coef, int64_t *count)
{
    const double PI2 = 2.0 * M_PI;
    const int nx = d->nx, ny = d->ny, nz = d->nz;
    const double tk = d->t0 + k * d->dt;
    const double rho = d->c * tk;                                  /* Alg. 4 */
    if (!(rho > 0)) return 0.0;
    /* S2 band rule (reading G11): the band's largest radius fixes the angles */
    const int b = k / kc->B;
    int kref = (b + 1) * kc->B - 1;
    if (kref > d->nt - 1) kref = d->nt - 1;
    const double rho_ref = d->c * (d->t0 + kref * d->dt);
    if (!(rho_ref > 0)) return 0.0;
    const double dtheta = kc->h / rho_ref;                          /* Eq. 37 */
    const double th_max = ref_theta_max(L, rho, kc->r_pad);         /* S9 */
    if (th_max < 0) return 0.0;
    double sum = 0.0;
    for (int i = 1;; ++i) {
        const double theta = i * dtheta;                            /* Eq. 38: theta_i = i dtheta */
        if (!(theta < M_PI)) break;
        if (theta > th_max) break;                                  /* S9: ring misses the padded box */
        const double st = sin(theta), ct = cos(theta);
        int64_t N; double dphi, omega;
        if (!d->literal) {                                          /* reading G2 */
            N = (int64_t)ceil(PI2 * rho_ref * st / kc->h);
            if (N < 1) N = 1;
            dphi = PI2 / (double)N;
            omega = st * dtheta * dphi;                             /* solid angle of the patch */
        } else {                                                    /* Eq. (37)-(38) as printed */
            dphi = kc->h / (rho_ref * st);
            N = (int64_t)floor(PI2 / dphi);
            omega = (kc->h * kc->h) / (rho_ref * rho_ref);
        }
        for (int64_t j = 0; j < N; ++j) {
            const double phi = (double)j * dphi;                    /* Eq. 38: phi_j = j dphi */
            const double cp = cos(phi), sp = sin(phi);
            double xi[3];
            for (int a = 0; a < 3; ++a) {
                const double u = st * cp * ex[a] + st * sp * ey[a] + ct * ez[a];    /* S3 */
                const double r = rq[a] + rho * u;                                     /* S4 */
                xi[a] = (r - d->origin[a]) / d->spacing;                              /* Alg. 4 */
            }
            if (xi[0] <= -1.0 || xi[0] >= nx || xi[1] <= -1.0 || xi[1] >= ny || xi[2] <= -1.0 || xi[2] >= nz)
                continue;                                           /* touches no node */
            const double fx0 = floor(xi[0]), fy0 = floor(xi[1]), fz0 = floor(xi[2]);
            const int ix = (int)fx0, iy = (int)fy0, iz = (int)fz0;
            const double fx = xi[0] - fx0, fy = xi[1] - fy0, fz = xi[2] - fz0;
            if (mode == 2) { ++*count; continue; }
            double val = 0.0;
            for (int cz = 0; cz < 2; ++cz) {
                const int z = iz + cz; if (z < 0 || z >= nz) continue;
                const double wz = cz ? fz : 1.0 - fz;               /* Eq. 10; Alg. 6 */
                for (int cy = 0; cy < 2; ++cy) {
                    const int y = iy + cy; if (y < 0 || y >= ny) continue;
                    const double wy = cy ? fy : 1.0 - fy;
                    for (int cx = 0; cx < 2; ++cx) {
                        const int xx = ix + cx; if (xx < 0 || xx >= nx) continue;
                        const double wx = cx ? fx : 1.0 - fx;
                        const int64_t n = ((int64_t)z * ny + y) * nx + xx;
                        if (mode == 0) val += wx * wy * wz * x[n];
                        else xs[n] += coef * omega * (wx * wy * wz);   /* S8 */
                    }
                }
            }
            sum += omega * val;
        }
    }
    return sum;
}

static void ref_set_threads(const oat_ref_desc *d)
{
#ifdef _OPENMP
    if (d->n_threads > 0) omp_set_num_threads(d->n_threads);
#else
    (void)d;
#endif
}

/* S5: g = G alpha, g[q*K+k] = rho_k^2 sum_ij omega A~(r_kij)   (Eq. 12, Eq. 36-38) */
int oat_ref_srt(const oat_ref_desc *d, const double *x, double *g)
{
    ref_consts kc; int rc = ref_setup(d, &kc); if (rc) return rc;
    if (!x || !g) return OAT_REF_ERR_INVALID;
    ref_set_threads(d);
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int q = 0; q < d->n_trans; ++q) {
        const double *rq = d->trans_xyz + 3 * (size_t)q;
        double ex[3], ey[3], ez[3], L;
        if (ref_frame(&kc, rq, ex, ey, ez, &L)) {
            _Pragma("omp atomic write")
            bad = 1;
            continue;
        }
        for (int k = 0; k < d->nt; ++k) {
            const double rho = d->c * (d->t0 + k * d->dt);
            const double s = ref_shell(d, &kc, rq, ex, ey, ez, L, k, 0, x, NULL, 0.0, NULL);
            g[(size_t)q * d->nt + k] = rho * rho * s;
        }
    }
    return bad ? OAT_REF_ERR_INVALID : OAT_REF_OK;
}

/* S8: alpha' = G^T g'   (Eq. 23; Alg. 6).  Transducers are summed in
 * index order within each thread; thread partial volumes are added in thread
 * order at the end. */
int oat_ref_srt_adjoint(const oat_ref_desc *d, const double *gp, double *x)
{
    ref_consts kc; int rc = ref_setup(d, &kc); if (rc) return rc;
    if (!gp || !x) return OAT_REF_ERR_INVALID;
    ref_set_threads(d);
    const size_t nvox = (size_t)d->nx * d->ny * d->nz;
    memset(x, 0, nvox * sizeof(double));
    int nth = 1;
#ifdef _OPENMP
    nth = omp_get_max_threads();
#endif
    if (nth > d->n_trans) nth = d->n_trans > 0 ? d->n_trans : 1;
    double *part = nth > 1 ? (double *)calloc(nvox * (size_t)nth, sizeof(double)) : x;
    if (!part) return OAT_REF_ERR_ALLOC;
    int bad = 0;
#pragma omp parallel num_threads(nth)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double *xs = part + nvox * (size_t)tid;
#pragma omp for schedule(static)
        for (int q = 0; q < d->n_trans; ++q) {
            const double *rq = d->trans_xyz + 3 * (size_t)q;
            double ex[3], ey[3], ez[3], L;
            if (ref_frame(&kc, rq, ex, ey, ez, &L)) {
            _Pragma("omp atomic write")
            bad = 1;
            continue;
        }
            for (int k = 0; k < d->nt; ++k) {
                const double gv = gp[(size_t)q * d->nt + k];
                if (gv == 0.0) continue;                           /* contributes exactly zero */
                const double rho = d->c * (d->t0 + k * d->dt);
                ref_shell(d, &kc, rq, ex, ey, ez, L, k, 1, NULL, xs, gv * rho * rho, NULL);
            }
        }
    }
    if (nth > 1) {
        for (int t = 0; t < nth; ++t)
            for (size_t n = 0; n < nvox; ++n) x[n] += part[nvox * (size_t)t + n];
        free(part);
    }
    return bad ? OAT_REF_ERR_INVALID : OAT_REF_OK;
}

/* S6: p = D g,  s_k = g_k/t_k,  p_k = kappa (s_{k+1} - s_{k-1}) / (2 dt)
 * (Eq. 3; Eq. 13 L125 with general t0; zero extension at both ends, G8; g/t := 0 at t <= 0, G9) */
int oat_ref_diff(const oat_ref_desc *d, const double *g, double *p)
{
    ref_consts kc; int rc = ref_setup(d, &kc); if (rc) return rc;
    if (!g || !p) return OAT_REF_ERR_INVALID;
    const int K = d->nt;
    for (int q = 0; q < d->n_trans; ++q) {
        const double *gq = g + (size_t)q * K; double *pq = p + (size_t)q * K;
        for (int k = 0; k < K; ++k) {
            double sp = 0.0, sm = 0.0;
            if (k + 1 < K) { double t = d->t0 + (k + 1) * d->dt; sp = t > 0 ? gq[k + 1] / t : 0.0; }
            if (k - 1 >= 0) { double t = d->t0 + (k - 1) * d->dt; sm = t > 0 ? gq[k - 1] / t : 0.0; }
            pq[k] = kc.kappa * (sp - sm) / (2.0 * d->dt);
        }
    }
    return OAT_REF_OK;
}

/* S7: g' = D^T y,  s'_k = kappa (y_{k-1} - y_{k+1}) / (2 dt),  g'_k = s'_k / t_k   (Eq. 22) */
int oat_ref_diff_adjoint(const oat_ref_desc *d, const double *y, double *gp)
{
    ref_consts kc; int rc = ref_setup(d, &kc); if (rc) return rc;
    if (!y || !gp) return OAT_REF_ERR_INVALID;
    const int K = d->nt;
    for (int q = 0; q < d->n_trans; ++q) {
        const double *yq = y + (size_t)q * K; double *gq = gp + (size_t)q * K;
        for (int k = 0; k < K; ++k) {
            const double ym = k - 1 >= 0 ? yq[k - 1] : 0.0;
            const double yp = k + 1 < K ? yq[k + 1] : 0.0;
            const double s = kc.kappa * (ym - yp) / (2.0 * d->dt);
            const double t = d->t0 + k * d->dt;
            gq[k] = t > 0 ? s / t : 0.0;
        }
    }
    return OAT_REF_OK;
}

/* H x = D (G x)   (Eq. 11 L116 without H^e) */
int oat_ref_project(const oat_ref_desc *d, const double *x, double *y)
{
    if (!d || d->nt <= 0 || d->n_trans < 0) return OAT_REF_ERR_INVALID;
    double *g = (double *)malloc(sizeof(double) * (size_t)(d->n_trans > 0 ? d->n_trans : 1) * d->nt);
    if (!g) return OAT_REF_ERR_ALLOC;
    int rc = oat_ref_srt(d, x, g);
    if (!rc) rc = oat_ref_diff(d, g, y);
    free(g);
    return rc;
}

/* H^T y = G^T (D^T y)   (L168: H^dagger = G^dagger D^dagger) */
int oat_ref_backproject(const oat_ref_desc *d, const double *y, double *x)
{
    if (!d || d->nt <= 0 || d->n_trans < 0) return OAT_REF_ERR_INVALID;
    double *gp = (double *)malloc(sizeof(double) * (size_t)(d->n_trans > 0 ? d->n_trans : 1) * d->nt);
    if (!gp) return OAT_REF_ERR_ALLOC;
    int rc = oat_ref_diff_adjoint(d, y, gp);
    if (!rc) rc = oat_ref_srt_adjoint(d, gp, x);
    free(gp);
    return rc;
}

/* Number of quadrature samples that fall inside the zero-padded node box, per
 * (q, k) if per_qk != NULL, and in total (the "interpolation samples" of the
 * throughput metric). */
int oat_ref_count_samples(const oat_ref_desc *d, int64_t *per_qk, int64_t *total)
{
    ref_consts kc; int rc = ref_setup(d, &kc); if (rc) return rc;
    ref_set_threads(d);
    int64_t tot = 0; int bad = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : tot)
    for (int q = 0; q < d->n_trans; ++q) {
        const double *rq = d->trans_xyz + 3 * (size_t)q;
        double ex[3], ey[3], ez[3], L;
        if (ref_frame(&kc, rq, ex, ey, ez, &L)) {
            _Pragma("omp atomic write")
            bad = 1;
            continue;
        }
        for (int k = 0; k < d->nt; ++k) {
            int64_t cnt = 0;
            ref_shell(d, &kc, rq, ex, ey, ez, L, k, 2, NULL, NULL, 0.0, &cnt);
            if (per_qk) per_qk[(size_t)q * d->nt + k] = cnt;
            tot += cnt;
        }
    }
    if (total) *total = tot;
    return bad ? OAT_REF_ERR_INVALID : OAT_REF_OK;
}

/* Sum of the quadrature's solid-angle weights over the WHOLE sphere for the
 * band that sample k belongs to (pin P3: -> 4 pi). */
int oat_ref_weight_sum(const oat_ref_desc *d, int k, double *wsum, int64_t *ndir)
{
    ref_consts kc; int rc = ref_setup(d, &kc); if (rc) return rc;
    if (k < 0 || k >= d->nt) return OAT_REF_ERR_INVALID;
    const int b = k / kc.B;
    int kref = (b + 1) * kc.B - 1; if (kref > d->nt - 1) kref = d->nt - 1;
    const double rho_ref = d->c * (d->t0 + kref * d->dt);
    if (!(rho_ref > 0)) return OAT_REF_ERR_INVALID;
    const double dtheta = kc.h / rho_ref;
    double s = 0; int64_t n = 0;
    for (int i = 1;; ++i) {
        const double theta = i * dtheta; if (!(theta < M_PI)) break;
        const double st = sin(theta);
        int64_t N; double omega;
        if (!d->literal) { N = (int64_t)ceil(2.0 * M_PI * rho_ref * st / kc.h); if (N < 1) N = 1; omega = st * dtheta * (2.0 * M_PI / (double)N); }
        else { N = (int64_t)floor(2.0 * M_PI / (kc.h / (rho_ref * st))); omega = kc.h * kc.h / (rho_ref * rho_ref); }
        s += omega * (double)N; n += N;
    }
    if (wsum) *wsum = s;
    if (ndir) *ndir = n;
    return OAT_REF_OK;
}

int oat_ref_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
