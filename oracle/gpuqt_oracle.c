/*
 * ORACLE — test infrastructure, NOT the product.
 *
 * A plain, slow, obviously-correct CPU implementation (fp64, C99) of what the GPUQT hot path
 * computes, written from the paper (/root/reference/PAPER.md = arXiv 1705.01387) equation by
 * equation.  No blocking, no fusion, no doubling identity, no reordering beyond what the
 * equations state; the only parallelism is an OpenMP "for" over rows.  It shares no code with the
 * CUDA library under paper_1705_01387_b200/csrc/ and neither includes the other.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call
 * this library.
 *
 * Parity pins (tests/test_oracle_pins.py, all -m "not gpu"): dense exact diagonalisation
 * (exp(-iHt), XU-UX, Tr T_n), plane-wave closed forms, Bessel identities and textbook values,
 * Jackson values computed from Eq. 31, Chebyshev-Gauss quadrature of the transform, clean-chain
 * DOS closed form.  The paper prints no numeric moment/DOS/conductivity value and its figures are
 * absent, so parity against the paper's own *results* is unpinned.
 *
 * Readings of silent/ambiguous points are marked [A#].
 *
 * Vectors are complex fp64 stored as interleaved (re, im) doubles, one vector = [N][2]; a batch is
 * [batch][N][2].
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_INDEX (-2)
#define ORACLE_ERR_ENERGY (-5)
#define ORACLE_ERR_NOMEM (-8)

typedef struct oracle_model {
    int64_t N;
    int32_t K;
    int32_t batch;
    int32_t *col;        /* [N*K] padded row-major; padding = (own row, hop 0)              */
    double *hre, *him;   /* [N*K] hopping H_{m,n_k}; Eq. 32                      */
    double *dx;          /* [N*K] minimum-image X_n - X_m  [A6]                               */
    double *onsite;      /* [N]   U_m                                                         */
    double *x;           /* [N]   X_m, Eq. 33                                    */
    double box, volume, dE;
    double *psi;         /* U(t) phi                      [batch][N][2]                       */
    double *chi;         /* [X, U(t)] phi                 [batch][N][2]  [A3]                 */
    double *va;          /* U(t)^dagger phi   (VAC bra)   [batch][N][2]  [A1]                 */
    double *vb;          /* U(t)^dagger V phi (VAC ket)   [batch][N][2]  [A1]                 */
} oracle_model;

/* ------------------------------------------------------------------ table */
static double min_image(double d, double box)
{
    /* [A6] d = X_n - X_m; wrap into (-L/2, L/2]; ties left unwrapped; box <= 0 => open boundary */
    if (box > 0.0) {
        if (d > 0.5 * box) d -= box;
        else if (d < -0.5 * box) d += box;
    }
    return d;
}

void oracle_destroy(oracle_model *m)
{
    if (!m) return;
    free(m->col); free(m->hre); free(m->him); free(m->dx); free(m->onsite); free(m->x);
    free(m->psi); free(m->chi); free(m->va); free(m->vb);
    free(m);
}

int oracle_create(oracle_model **out, int64_t N, int32_t K, const int32_t *nbr_count,
                  const int32_t *nbr_index, const double *hop_re, const double *hop_im,
                  const double *onsite, const double *x, double box_length, double volume,
                  double energy_scale, int32_t batch)
{
    if (!out || N <= 0 || K <= 0 || !nbr_count || !nbr_index || !x || batch <= 0 ||
        !(energy_scale > 0.0))
        return ORACLE_ERR_ARG;
    oracle_model *m = (oracle_model *)calloc(1, sizeof(*m));
    if (!m) return ORACLE_ERR_NOMEM;
    m->N = N; m->K = K; m->batch = batch;
    m->box = box_length; m->volume = volume; m->dE = energy_scale;
    size_t nk = (size_t)N * (size_t)K, nv = (size_t)batch * (size_t)N * 2;
    m->col = (int32_t *)malloc(nk * sizeof(int32_t));
    m->hre = (double *)malloc(nk * sizeof(double));
    m->him = (double *)malloc(nk * sizeof(double));
    m->dx = (double *)malloc(nk * sizeof(double));
    m->onsite = (double *)malloc((size_t)N * sizeof(double));
    m->x = (double *)malloc((size_t)N * sizeof(double));
    m->psi = (double *)calloc(nv, sizeof(double));
    m->chi = (double *)calloc(nv, sizeof(double));
    m->va = (double *)calloc(nv, sizeof(double));
    m->vb = (double *)calloc(nv, sizeof(double));
    if (!m->col || !m->hre || !m->him || !m->dx || !m->onsite || !m->x || !m->psi || !m->chi ||
        !m->va || !m->vb) { oracle_destroy(m); return ORACLE_ERR_NOMEM; }
    for (int64_t r = 0; r < N; ++r) {
        m->x[r] = x[r];
        m->onsite[r] = onsite ? onsite[r] : 0.0;               /* default 0 */
    }
    for (int64_t r = 0; r < N; ++r) {
        int32_t c = nbr_count[r];
        if (c < 0 || c > K) { oracle_destroy(m); return ORACLE_ERR_INDEX; }
        for (int32_t k = 0; k < K; ++k) {
            size_t e = (size_t)r * K + k;
            if (k < c) {
                int32_t n = nbr_index[e];                      /* 0-based [A11] */
                if (n < 0 || n >= N) { oracle_destroy(m); return ORACLE_ERR_INDEX; }
                m->col[e] = n;
                m->hre[e] = hop_re ? hop_re[e] : -1.0;         /* default -1 */
                m->him[e] = hop_im ? hop_im[e] : 0.0;
                m->dx[e] = min_image(x[n] - x[r], box_length);
            } else {
                m->col[e] = (int32_t)r; m->hre[e] = 0.0; m->him[e] = 0.0; m->dx[e] = 0.0;
            }
        }
    }
    *out = m;
    return ORACLE_OK;
}

/* canonical padded table for the bit-exact indexing comparison */
int oracle_get_table(const oracle_model *m, int32_t *col, double *re, double *im, double *dx)
{
    size_t nk = (size_t)m->N * m->K;
    if (col) memcpy(col, m->col, nk * sizeof(int32_t));
    if (re) memcpy(re, m->hre, nk * sizeof(double));
    if (im) memcpy(im, m->him, nk * sizeof(double));
    if (dx) memcpy(dx, m->dx, nk * sizeof(double));
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ operators (step 2) */
/* out = H~ in = (U_m in_m + sum_k H_{m,n_k} in_{n_k}) / dE      PAPER.md:231 Eq. 32, :160 Eq. 19 */
int oracle_apply_h(const oracle_model *m, const double *in, double *out)
{
    const int64_t N = m->N; const int32_t K = m->K;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < N; ++r) {
        double sr = m->onsite[r] * in[2 * r], si = m->onsite[r] * in[2 * r + 1];
        for (int32_t k = 0; k < K; ++k) {
            size_t e = (size_t)r * K + k;
            int64_t n = m->col[e];
            double hr = m->hre[e], hi = m->him[e];
            double vr = in[2 * n], vi = in[2 * n + 1];
            sr += hr * vr - hi * vi;
            si += hr * vi + hi * vr;
        }
        out[2 * r] = sr / m->dE;
        out[2 * r + 1] = si / m->dE;
    }
    return ORACLE_OK;
}

/* out = V in,  V_mn = (i/hbar)(X_n - X_m) H_mn, hbar = 1       PAPER.md:237 Eq. 34 [A2][A8]
 * not divided by dE; no on-site term (X_m - X_m = 0)                                          */
int oracle_apply_v(const oracle_model *m, const double *in, double *out)
{
    const int64_t N = m->N; const int32_t K = m->K;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < N; ++r) {
        double sr = 0.0, si = 0.0;
        for (int32_t k = 0; k < K; ++k) {
            size_t e = (size_t)r * K + k;
            int64_t n = m->col[e];
            double wr = m->dx[e] * m->hre[e], wi = m->dx[e] * m->him[e];   /* (X_n - X_m) H_mn */
            double vr = in[2 * n], vi = in[2 * n + 1];
            sr += wr * vr - wi * vi;
            si += wr * vi + wi * vr;
        }
        out[2 * r] = -si;            /* multiply by i: i (sr + i si) = -si + i sr */
        out[2 * r + 1] = sr;
    }
    return ORACLE_OK;
}

/* out = [X, H~] in,  [X,H~]_mn = (X_m - X_n) H_mn / dE           (from Eq. 33, 19) */
int oracle_apply_xh(const oracle_model *m, const double *in, double *out)
{
    const int64_t N = m->N; const int32_t K = m->K;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < N; ++r) {
        double sr = 0.0, si = 0.0;
        for (int32_t k = 0; k < K; ++k) {
            size_t e = (size_t)r * K + k;
            int64_t n = m->col[e];
            double wr = -m->dx[e] * m->hre[e], wi = -m->dx[e] * m->him[e];  /* (X_m - X_n) H_mn */
            double vr = in[2 * n], vi = in[2 * n + 1];
            sr += wr * vr - wi * vi;
            si += wr * vi + wi * vr;
        }
        out[2 * r] = sr / m->dE;
        out[2 * r + 1] = si / m->dE;
    }
    return ORACLE_OK;
}

/* <l|r> = sum conj(l_i) r_i, accumulated in long double */
static void dot(int64_t N, const double *l, const double *r, double *re, double *im)
{
    long double sr = 0.0L, si = 0.0L;
#pragma omp parallel for schedule(static) reduction(+ : sr, si)
    for (int64_t i = 0; i < N; ++i) {
        long double lr = l[2 * i], li = l[2 * i + 1], rr = r[2 * i], ri = r[2 * i + 1];
        sr += lr * rr + li * ri;
        si += lr * ri - li * rr;
    }
    *re = (double)sr; *im = (double)si;
}

/* ------------------------------------------------------------------ Bessel coefficients (step 3) */
/* c_m = (2 - delta_{0m}) (-+ i)^m J_m(dE |dt|) for U(+-|dt|)      PAPER.md:154 Eq. 17, :162 Eq. 20 */
int oracle_bessel_coeffs(double dE, double dt, int32_t order, double *c_re, double *c_im)
{
    double arg = dE * fabs(dt);                                 /* hbar = 1 [A8] */
    int sgn = dt < 0 ? -1 : 1;
    for (int32_t k = 0; k < order; ++k) {
        double j = jn(k, arg) * (k == 0 ? 1.0 : 2.0);
        /* (-i sgn)^k : k mod 4 = 0: 1, 1: -i sgn, 2: -1, 3: +i sgn */
        switch (k & 3) {
        case 0: c_re[k] = j; c_im[k] = 0.0; break;
        case 1: c_re[k] = 0.0; c_im[k] = -sgn * j; break;
        case 2: c_re[k] = -j; c_im[k] = 0.0; break;
        default: c_re[k] = 0.0; c_im[k] = sgn * j; break;
        }
    }
    return ORACLE_OK;
}

static void axpy_c(int64_t N, double cr, double ci, const double *v, double *acc)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
        double vr = v[2 * i], vi = v[2 * i + 1];
        acc[2 * i] += cr * vr - ci * vi;
        acc[2 * i + 1] += cr * vi + ci * vr;
    }
}

/* out = sum_{k<order} c_k T_k(H~) in, forward recurrence Eq. 21/23 then the sum Eq. 17
 * — separate loops (step 4).                                          */
int oracle_evolve_vec(const oracle_model *m, const double *in, double *out, double dt,
                      int32_t order)
{
    const int64_t N = m->N;
    if (order < 1) return ORACLE_ERR_ARG;
    size_t bytes = (size_t)N * 2 * sizeof(double);
    double *cr = (double *)malloc(order * sizeof(double)), *ci = (double *)malloc(order * sizeof(double));
    double *t0 = (double *)malloc(bytes), *t1 = (double *)malloc(bytes), *t2 = (double *)malloc(bytes);
    double *acc = (double *)calloc((size_t)N * 2, sizeof(double));
    if (!cr || !ci || !t0 || !t1 || !t2 || !acc) { free(cr); free(ci); free(t0); free(t1); free(t2); free(acc); return ORACLE_ERR_NOMEM; }
    oracle_bessel_coeffs(m->dE, dt, order, cr, ci);
    memcpy(t0, in, bytes);                                       /* T_0 in = in   (Eq. 23) */
    axpy_c(N, cr[0], ci[0], t0, acc);
    if (order > 1) {
        oracle_apply_h(m, t0, t1);                               /* T_1 in = H~ in (Eq. 23) */
        axpy_c(N, cr[1], ci[1], t1, acc);
    }
    for (int32_t k = 2; k < order; ++k) {
        oracle_apply_h(m, t1, t2);                               /* T_k = 2 H~ T_{k-1} - T_{k-2} */
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < 2 * N; ++i) t2[i] = 2.0 * t2[i] - t0[i];
        axpy_c(N, cr[k], ci[k], t2, acc);
        double *tmp = t0; t0 = t1; t1 = t2; t2 = tmp;
    }
    memcpy(out, acc, bytes);
    free(cr); free(ci); free(t0); free(t1); free(t2); free(acc);
    return ORACLE_OK;
}

/* out = [X, U(dt)] in = sum_k c_k [X, T_k] in                       PAPER.md:156 Eq. 18
 * a_k = T_k in (Eq. 21, 23);  b_k = [X,T_k] in:  b_0 = 0, b_1 = [X,H~] in (Eq. 24),
 * b_k = 2 [X,H~] a_{k-1} + 2 H~ b_{k-1} - b_{k-2}                    (Eq. 22)  (step 5)        */
int oracle_commutator_vec(const oracle_model *m, const double *in, double *out, double dt,
                          int32_t order)
{
    const int64_t N = m->N;
    if (order < 1) return ORACLE_ERR_ARG;
    size_t bytes = (size_t)N * 2 * sizeof(double);
    double *cr = (double *)malloc(order * sizeof(double)), *ci = (double *)malloc(order * sizeof(double));
    double *a0 = (double *)malloc(bytes), *a1 = (double *)malloc(bytes), *a2 = (double *)malloc(bytes);
    double *b0 = (double *)calloc((size_t)N * 2, sizeof(double)), *b1 = (double *)malloc(bytes), *b2 = (double *)malloc(bytes);
    double *w1 = (double *)malloc(bytes), *w2 = (double *)malloc(bytes);
    double *acc = (double *)calloc((size_t)N * 2, sizeof(double));
    if (!cr || !ci || !a0 || !a1 || !a2 || !b0 || !b1 || !b2 || !w1 || !w2 || !acc) {
        free(cr); free(ci); free(a0); free(a1); free(a2); free(b0); free(b1); free(b2); free(w1); free(w2); free(acc);
        return ORACLE_ERR_NOMEM;
    }
    oracle_bessel_coeffs(m->dE, dt, order, cr, ci);
    memcpy(a0, in, bytes);                                       /* a_0 = in; b_0 = 0 */
    if (order > 1) {
        oracle_apply_h(m, a0, a1);                               /* a_1 = H~ in        */
        oracle_apply_xh(m, a0, b1);                              /* b_1 = [X,H~] in    */
        axpy_c(N, cr[1], ci[1], b1, acc);
    }
    for (int32_t k = 2; k < order; ++k) {
        oracle_apply_xh(m, a1, w1);                              /* [X,H~] a_{k-1} */
        oracle_apply_h(m, b1, w2);                               /* H~ b_{k-1}     */
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < 2 * N; ++i) b2[i] = 2.0 * w1[i] + 2.0 * w2[i] - b0[i];
        axpy_c(N, cr[k], ci[k], b2, acc);
        oracle_apply_h(m, a1, a2);                               /* a_k = 2 H~ a_{k-1} - a_{k-2} */
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < 2 * N; ++i) a2[i] = 2.0 * a2[i] - a0[i];
        double *t = a0; a0 = a1; a1 = a2; a2 = t;
        t = b0; b0 = b1; b1 = b2; b2 = t;
    }
    memcpy(out, acc, bytes);
    free(cr); free(ci); free(a0); free(a1); free(a2); free(b0); free(b1); free(b2); free(w1); free(w2); free(acc);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ state and time stepping */
/* phi: host [batch][N][2].  psi = phi, chi = 0 ([X,U(0)] = 0), a = phi, b = V phi  [A1][A3] */
int oracle_set_state(oracle_model *m, const double *phi)
{
    size_t nv = (size_t)m->batch * m->N * 2;
    memcpy(m->psi, phi, nv * sizeof(double));
    memset(m->chi, 0, nv * sizeof(double));
    memcpy(m->va, phi, nv * sizeof(double));
    for (int32_t b = 0; b < m->batch; ++b)
        oracle_apply_v(m, phi + (size_t)b * m->N * 2, m->vb + (size_t)b * m->N * 2);
    return ORACLE_OK;
}

#define ORACLE_MODE_VAC 1
#define ORACLE_MODE_MSD 2

/* One time step of every enabled branch (steps 5, 6):
 *   psi' = U(dt) psi
 *   chi' = U(dt) chi + [X,U(dt)] psi    (product rule [X,U2 U1] = [X,U2]U1 + U2[X,U1])  [A3]
 *   a'   = U(-dt) a,  b' = U(-dt) b     (Eq. 29: the ket is U(t)^dagger V phi)          [A1]   */
int oracle_evolve(oracle_model *m, double dt, int32_t order, int modes)
{
    const int64_t N = m->N;
    size_t bytes = (size_t)N * 2 * sizeof(double);
    double *u = (double *)malloc(bytes), *c = (double *)malloc(bytes);
    if (!u || !c) { free(u); free(c); return ORACLE_ERR_NOMEM; }
    int rc = ORACLE_OK;
    for (int32_t b = 0; b < m->batch && rc == ORACLE_OK; ++b) {
        double *psi = m->psi + (size_t)b * N * 2, *chi = m->chi + (size_t)b * N * 2;
        double *va = m->va + (size_t)b * N * 2, *vb = m->vb + (size_t)b * N * 2;
        if (modes & ORACLE_MODE_MSD) {
            rc = oracle_evolve_vec(m, chi, u, dt, order);                 /* U chi       */
            if (rc) break;
            rc = oracle_commutator_vec(m, psi, c, dt, order);             /* [X,U] psi   */
            if (rc) break;
            for (int64_t i = 0; i < 2 * N; ++i) chi[i] = u[i] + c[i];
        }
        rc = oracle_evolve_vec(m, psi, u, dt, order);                     /* U psi       */
        if (rc) break;
        memcpy(psi, u, bytes);
        if (modes & ORACLE_MODE_VAC) {
            rc = oracle_evolve_vec(m, va, u, -dt, order);
            if (rc) break;
            memcpy(va, u, bytes);
            rc = oracle_evolve_vec(m, vb, u, -dt, order);
            if (rc) break;
            memcpy(vb, u, bytes);
        }
    }
    free(u); free(c);
    return rc;
}

/* which: 0 psi, 1 chi, 2 a, 3 b */
int oracle_get_state(const oracle_model *m, int which, double *out)
{
    const double *src = which == 0 ? m->psi : which == 1 ? m->chi : which == 2 ? m->va : which == 3 ? m->vb : NULL;
    if (!src) return ORACLE_ERR_ARG;
    memcpy(out, src, (size_t)m->batch * m->N * 2 * sizeof(double));
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ moments (step 7) */
/* C_n = <l| T_n(H~) |r>, n < n_moments, by the plain definition: r_0 = r, r_1 = H~ r,
 * r_n = 2 H~ r_{n-1} - r_{n-2}  (Eq. 21, 23); no doubling identity.          */
int oracle_moments_vec(const oracle_model *m, const double *l, const double *r, int32_t n_moments,
                       double *c_re, double *c_im)
{
    const int64_t N = m->N;
    size_t bytes = (size_t)N * 2 * sizeof(double);
    double *t0 = (double *)malloc(bytes), *t1 = (double *)malloc(bytes), *t2 = (double *)malloc(bytes);
    if (!t0 || !t1 || !t2) { free(t0); free(t1); free(t2); return ORACLE_ERR_NOMEM; }
    double re, im;
    memcpy(t0, r, bytes);
    if (n_moments > 0) { dot(N, l, t0, &re, &im); c_re[0] = re; if (c_im) c_im[0] = im; }
    if (n_moments > 1) {
        oracle_apply_h(m, t0, t1);
        dot(N, l, t1, &re, &im); c_re[1] = re; if (c_im) c_im[1] = im;
    }
    for (int32_t n = 2; n < n_moments; ++n) {
        oracle_apply_h(m, t1, t2);
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < 2 * N; ++i) t2[i] = 2.0 * t2[i] - t0[i];
        dot(N, l, t2, &re, &im); c_re[n] = re; if (c_im) c_im[n] = im;
        double *t = t0; t0 = t1; t1 = t2; t2 = t;
    }
    free(t0); free(t1); free(t2);
    return ORACLE_OK;
}

/* C_n^DOS = <phi|T_n|phi>, phi = the vector given at set_state; we keep it as a(0)... the DOS is
 * time independent, so it is evaluated on psi at the current time: <psi|T_n|psi> = <phi|T_n|phi>
 * only at t = 0 in floating point; callers take it before evolving.   PAPER.md:192 Eq. 28 [A16] */
int oracle_dos_moments(const oracle_model *m, int32_t n_moments, double *out /* [batch][n] */)
{
    for (int32_t b = 0; b < m->batch; ++b) {
        const double *v = m->psi + (size_t)b * m->N * 2;
        int rc = oracle_moments_vec(m, v, v, n_moments, out + (size_t)b * n_moments, NULL);
        if (rc) return rc;
    }
    return ORACLE_OK;
}

/* C_n^MSD(t) = <phi|[X,U]^dagger T_n [X,U]|phi> = <chi|T_n|chi>      PAPER.md:198 Eq. 30 [A16] */
int oracle_msd(const oracle_model *m, int32_t n_moments, double *out)
{
    for (int32_t b = 0; b < m->batch; ++b) {
        const double *v = m->chi + (size_t)b * m->N * 2;
        int rc = oracle_moments_vec(m, v, v, n_moments, out + (size_t)b * n_moments, NULL);
        if (rc) return rc;
    }
    return ORACLE_OK;
}

/* C_n^VAC(t) = Re <phi|U V T_n U^dagger V|phi> = Re <V a|T_n|b>, a = U^dagger phi,
 * b = U^dagger V phi (V Hermitian: <phi|U V = (V U^dagger phi)^dagger)  PAPER.md:195 Eq. 29 [A1] */
int oracle_vac(const oracle_model *m, int32_t n_moments, double *out)
{
    size_t bytes = (size_t)m->N * 2 * sizeof(double);
    double *l = (double *)malloc(bytes);
    if (!l) return ORACLE_ERR_NOMEM;
    for (int32_t b = 0; b < m->batch; ++b) {
        oracle_apply_v(m, m->va + (size_t)b * m->N * 2, l);
        int rc = oracle_moments_vec(m, l, m->vb + (size_t)b * m->N * 2, n_moments,
                                    out + (size_t)b * n_moments, NULL);
        if (rc) { free(l); return rc; }
    }
    free(l);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ Jackson + transform (step 8) */
/* g_n = (1 - n alpha) cos(pi n alpha) + alpha sin(pi n alpha) cot(pi alpha), alpha = 1/(N_m+1)
 * PAPER.md:203 Eq. 31 [A14]                                                                    */
int oracle_jackson(int32_t n_moments, double *g)
{
    double alpha = 1.0 / ((double)n_moments + 1.0);
    for (int32_t n = 0; n < n_moments; ++n)
        g[n] = (1.0 - n * alpha) * cos(M_PI * n * alpha) +
               alpha * sin(M_PI * n * alpha) / tan(M_PI * alpha);
    return ORACLE_OK;
}

/* Other damping kernels of the kernel polynomial method (the paper's ref. [33]; the paper
 * itself uses Jackson only -- SURVEY.md 8(f) 5):
 *   kind 0  Jackson, Eq. 31
 *   kind 1  Lorentz:  g_n = sinh(lambda (1 - n / N_m)) / sinh(lambda), lambda > 0
 *           (turns delta(x - a) into a Lorentzian of half width lambda / N_m in the rescaled variable)
 *   kind 2  none (Dirichlet):  g_n = 1, the plain truncated Chebyshev series                        */
int oracle_damping(int kind, double lambda, int32_t n_moments, double *g)
{
    if (kind == 0) return oracle_jackson(n_moments, g);
    if (kind == 1) {
        if (!(lambda > 0.0)) return ORACLE_ERR_ARG;
        for (int32_t n = 0; n < n_moments; ++n)
            g[n] = sinh(lambda * (1.0 - (double)n / (double)n_moments)) / sinh(lambda);
        return ORACLE_OK;
    }
    if (kind == 2) {
        for (int32_t n = 0; n < n_moments; ++n) g[n] = 1.0;
        return ORACLE_OK;
    }
    return ORACLE_ERR_ARG;
}

/* out[s][j] = 2 / (pi Omega dE sqrt(1 - E~^2)) sum_n g_n (2 - delta_n0) T_n(E~) C_n[s]
 * with E~ = E_j / dE and T_n(E~) = cos(n arccos E~).     PAPER.md:184-188 Eq. 25-27 [A15][A21] */
int oracle_kpm_transform_damped(const oracle_model *m, int kind, double lambda, const double *moments,
                                int32_t n_moments, int32_t n_sets, const double *energies,
                                int32_t n_energies, double *out)
{
    double *g = (double *)malloc((size_t)n_moments * sizeof(double));
    if (!g) return ORACLE_ERR_NOMEM;
    int rc = oracle_damping(kind, lambda, n_moments, g);
    if (rc != ORACLE_OK) { free(g); return rc; }
    for (int32_t j = 0; j < n_energies; ++j)
        if (!(fabs(energies[j] / m->dE) < 1.0)) { free(g); return ORACLE_ERR_ENERGY; }
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < n_energies; ++j) {
        double e = energies[j] / m->dE, th = acos(e);
        double pref = 2.0 / (M_PI * m->volume * m->dE * sqrt(1.0 - e * e));
        for (int32_t s = 0; s < n_sets; ++s) {
            long double sum = 0.0L;
            for (int32_t n = 0; n < n_moments; ++n)
                sum += (long double)(g[n] * (n == 0 ? 1.0 : 2.0) * cos(n * th)) *
                       moments[(size_t)s * n_moments + n];
            out[(size_t)s * n_energies + j] = pref * (double)sum;
        }
    }
    free(g);
    return ORACLE_OK;
}

int oracle_kpm_transform(const oracle_model *m, const double *moments, int32_t n_moments,
                         int32_t n_sets, const double *energies, int32_t n_energies, double *out)
{
    return oracle_kpm_transform_damped(m, 0, 0.0, moments, n_moments, n_sets, energies, n_energies, out);
}

/* Running conductivity from the transformed correlation functions (units e = 1), Eq. 2,
 * :92 Eq. 5, :123 Eq. 11; discretisation readings [A25][A26] of DESIGN.md:
 *   kind 0 (VAC)  in[k][j] = rho(E_j) C_vv(E_j, t_k), rows at t_k = sum_{i<k} dt_i  (measure, evolve [A4]);
 *                 sigma[k][j] = int_0^{t_k} rho C_vv dt by the trapezoid rule, sigma[0][j] = 0.
 *   kind 1 (MSD)  in[k][j] = rho(E_j) dX^2(E_j, t_{k+1}), rows at t_{k+1} = sum_{i<=k} dt_i (evolve, measure),
 *                 dX^2(t = 0) = 0;  sigma[k][j] = (in[k][j] - in[k-1][j]) / (2 dt_k): the time derivative of
 *                 Eq. 5 by the difference over step k, i.e. the running conductivity at the MIDDLE of step k;
 *                 length[k][j] = 2 sqrt(in[k][j] / dos[j])  (Eq. 11; 0 where dos <= 0 or in < 0).
 * dos[j] = rho(E_j) (Eq. 4) is used for the length only; length may be NULL.                      */
int oracle_running_conductivity(int kind, const double *in, const double *dos, const double *dt,
                                int32_t n_t, int32_t n_e, double *sigma, double *length)
{
    if (!in || !dt || !sigma || n_t < 1 || n_e < 1 || (kind != 0 && kind != 1)) return ORACLE_ERR_ARG;
    for (int32_t j = 0; j < n_e; ++j) {
        if (kind == 0) {
            double acc = 0.0;
            sigma[j] = 0.0;
            for (int32_t k = 1; k < n_t; ++k) {
                acc += 0.5 * (in[(size_t)(k - 1) * n_e + j] + in[(size_t)k * n_e + j]) * dt[k - 1];
                sigma[(size_t)k * n_e + j] = acc;
            }
        } else {
            for (int32_t k = 0; k < n_t; ++k) {
                double now = in[(size_t)k * n_e + j];
                double before = k > 0 ? in[(size_t)(k - 1) * n_e + j] : 0.0;
                sigma[(size_t)k * n_e + j] = (now - before) / (2.0 * dt[k]);
                if (length) {
                    double r = (dos && dos[j] > 0.0 && now > 0.0) ? now / dos[j] : 0.0;
                    length[(size_t)k * n_e + j] = 2.0 * sqrt(r);
                }
            }
        }
    }
    return ORACLE_OK;
}

/* Localization length from the propagating length (Eq. 12):  xi(E_j) = lim_t L(E_j, t) / (2 pi).
 * The limit is read as the LAST measured time [A27]:  xi[j] = length[n_t - 1][j] / (2 pi), and the saturation that
 * Eq. 12 presupposes ("the propagating length will finally saturate") is reported beside it as the
 * relative change of L over the last step,  growth[j] = (L[n_t-1][j] - L[n_t-2][j]) / L[n_t-1][j]
 * (0 where L[n_t-1][j] == 0; 1 when there is only one row: nothing is known about saturation).  growth may be NULL. */
int oracle_localization_length(const double *length, int32_t n_t, int32_t n_e, double *xi, double *growth)
{
    if (!length || !xi || n_t < 1 || n_e < 1) return ORACLE_ERR_ARG;
    const double two_pi = 2.0 * 3.14159265358979323846;
    for (int32_t j = 0; j < n_e; ++j) {
        double last = length[(size_t)(n_t - 1) * n_e + j];
        xi[j] = last / two_pi;
        if (growth) {
            if (last == 0.0) growth[j] = 0.0;
            else if (n_t == 1) growth[j] = 1.0;
            else growth[j] = (last - length[(size_t)(n_t - 2) * n_e + j]) / last;
        }
    }
    return ORACLE_OK;
}
