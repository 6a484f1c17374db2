/*
 * heat_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU implementation of one time step of the
 * explicit-implicit finite-difference scheme of arXiv 1408.5853 (Ayriyan et al.),
 * written from the paper step by step in the paper's order and notation.
 * "P:Lnnn" cites a line of /root/reference/PAPER.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this file.  It shares no code with the CUDA path
 * (paper_1408_5853_b200/csrc) and neither includes the other.
 *
 * Arithmetic: ORC_REAL (double by default; -DORC_LONG_DOUBLE builds the same code in
 * x87 extended precision for the rounding-floor estimate).  No blocking, fusion or
 * reordering beyond what the paper's formulas state.  The only parallel construct is an
 * optional `#pragma omp parallel for` over the line index j (the paper's own
 * decomposition): lines are independent within a step, so the result is
 * bitwise identical to the serial build.
 *
 * Readings of garbled / silent passages:
 *   G1  (10) prefactor is 1/(r_i hbar_i)            G2  (11) prefactor is 1/etabar_j
 *   G3  lambda_{i+-1/2} = lambda_m((T_a+T_b)/2) [face_mode 0]; mean of lambdas [face_mode 1]
 *   G7  (18) second line is at the new level        G8  (22) exponent is negative
 *   G9  source sampled at the start of the step     G14 material belongs to r-segments
 *   G16 Neumann z-line copies its neighbour         G17 Dirichlet z-lines are never solved
 *   G24 non-rectangular Omega, "N_j" of (9) P:L117 and Fig. 1: a stepped domain -- the lines above z_{j_step}
 *       end at node i_step (the core reaching the terminal) with zero flux (6) on the two new faces
 *   G23 (variant orc_step_picard only) "iterations at each time step" P:L206 = simple iteration on
 *       the coefficients: laws at the previous iterate, the current level where (8) has it
 *
 * Pins: tests/test_oracle_*.py (dense solve, discrete steady state, ln r, z-sine growth
 * factor, Bessel mode, lumped heating, energy identity, interface flux, schedule table,
 * tau-consistency with P:L278/L322) and, since round 2, tests/test_oracle_pins_r2.py: rows (13)
 * re-assembled in NumPy (both face modes), the face_mode-1 rule on a hand-computed line and in
 * the energy identity, probe records against the field of their step (bitwise);
 * tests/test_oracle_picard.py for orc_step_picard (bitwise the paper's step for one iteration and
 * for T-independent laws, a NumPy residual of the rows with the laws at the previous iterate, the
 * fixed point).  Every function here has a pin.  What the PAPER cannot decide (both sides take the same reading): which of the
 * two face rules G3 it means, and G9.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORC_LONG_DOUBLE
typedef long double real;
#define R_POW powl
#define R_EXP expl
#else
typedef double real;
#define R_POW pow
#define R_EXP exp
#endif

enum { ORC_LAW_CONST = 0, ORC_LAW_POWER = 1, ORC_LAW_POLY = 2 };
enum { ORC_BC_NEUMANN0 = 0, ORC_BC_DIRICHLET = 1 };

typedef struct {
    int32_t kind;
    int32_t pad_;
    double c[5];   /* CONST: c[0]; POWER: c[0]*(T/T_ref)^c[1]; POLY: sum_k c[k] T^k (23),(24) */
    double T_ref;
} orc_law;

typedef struct {
    orc_law k;          /* lambda_m(T), eq.(1) */
    orc_law cp;         /* c_Vm(T) */
    double rho;         /* rho_m */
    int32_t is_heater;  /* X_m != 0 only here */
    int32_t pad_;
    orc_law src_shape;  /* s(T): X = Q0 * s(T) * nu(t) p^2(t); chi(T) of (25) up to a constant */
} orc_layer;

typedef struct {
    int32_t kind;
    int32_t pad_;
    double value;
} orc_bc;

typedef struct {
    int32_t nr, nz, batch, nlayers;
    const double *r, *z;             /* node coordinates, ascending (9) P:L117 */
    const orc_layer *layers;
    const uint8_t *seg_layer;        /* batch*(nr-1): layer of radial segment (i,i+1), G14 */
    orc_bc r_in, r_out, z_lo, z_hi;  /* (6) P:L90-95, generalised per side */
    double T0;                       /* (5) P:L86 */
    const double *T_init;            /* optional batch*nz*nr, r fastest */
    double dt;                       /* tau */
    const double *Q0;                /* batch: source amplitude */
    int64_t steps_per_period;        /* t_prd / tau  (4) P:L79; 0 = no source */
    int64_t steps_on;                /* t_src / tau */
    int32_t transient_substeps;      /* 100 in the paper; 0 = Heaviside p(t) */
    int32_t face_mode;               /* G3 */
    double transient_k;              /* 7 in the paper */
    int32_t nprobes, probe_every;
    const int32_t *probe_ij;         /* nprobes*(i,j) */
    int32_t i_step, j_step;          /* stepped domain (G24): lines j > j_step end at node i_step; 0, 0 = rectangle */
} orc_desc;

typedef struct {
    int nr, nz, batch, nlayers;
    double *r, *z;
    orc_layer *layers;
    uint8_t *seg_layer;
    orc_bc r_in, r_out, z_lo, z_hi;
    double dt;
    double *Q0;
    int64_t steps_per_period, steps_on;
    int transient_substeps, face_mode;
    double transient_k;
    int nprobes, probe_every;
    int32_t *probe_ij;
    int i_step, j_step;
    /* state */
    real *T, *Tn;       /* two time levels, [batch][nz][nr], r fastest */
    real *Ts;           /* iterate of the new level (orc_step_picard only; allocated on first use) */
    real *alpha, *beta; /* sweep coefficients, one line per j (nz*nr) so that lines are independent */
    int64_t step;       /* solver steps done */
    double *probe;      /* growable: batch*nprobes values per record */
    int64_t probe_len, probe_cap;
} orc_ctx;

/* ------------------------------------------------------------------ laws */

static real law_eval(const orc_law *L, real T)
{
    switch (L->kind) {
    case ORC_LAW_CONST:
        return (real)L->c[0];
    case ORC_LAW_POWER:
        return (real)L->c[0] * R_POW(T / (real)L->T_ref, (real)L->c[1]);
    default: { /* ORC_LAW_POLY: sum_{k=0}^{4} c_k T^k, eqs. (23),(24) P:L245-248 */
        real s = 0, p = 1;
        for (int k = 0; k < 5; ++k) {
            s += (real)L->c[k] * p;
            p *= T;
        }
        return s;
    }
    }
}

/* lambda at a half node, P:L127 (reading G3) */
static real face_lambda(const orc_ctx *c, const orc_law *k, real Ta, real Tb)
{
    if (c->face_mode == 0)
        return law_eval(k, (Ta + Tb) / 2);
    return (law_eval(k, Ta) + law_eval(k, Tb)) / 2;
}

/* ------------------------------------------------------------------ schedule */

/* Step schedule, eqs. (4) P:L79 and (22) + procedure P:L212-217, integer counters only (G18).
 * Solver step s (0-based).  With the transient model the first step of every period is
 * replaced by `transient_substeps` sub-steps of tau* = tau/transient_substeps with
 * p^2 = 1 - exp(-q/transient_k) at sub-step q (time sampled at the start of the step, G9);
 * afterwards steps of tau with p^2 = 1; nu = 1 while (step in period) < steps_on. */
void orc_schedule(const orc_ctx *c, int64_t s, double *tau, double *amp)
{
    int64_t P = c->steps_per_period, S = c->steps_on;
    int nsub = c->transient_substeps;
    if (P <= 0 || S <= 0) {
        *tau = c->dt;
        *amp = 0.0;
        return;
    }
    if (nsub > 0) {
        int64_t L = (int64_t)nsub + P - 1; /* solver steps per period */
        int64_t q = s % L;
        if (q < nsub) {
            *tau = c->dt / (double)nsub;
            *amp = 1.0 - exp(-(double)q / c->transient_k);
        } else {
            int64_t g = q - nsub + 1; /* index of the tau-step inside the period, 1..P-1 */
            *tau = c->dt;
            *amp = (g < S) ? 1.0 : 0.0;
        }
    } else {
        int64_t g = s % P;
        *tau = c->dt;
        *amp = (g < S) ? 1.0 : 0.0;
    }
}

/* ------------------------------------------------------------------ rows */

/* Coefficients (13) P:L140-145 of a regular node (i,j), layer m, from the current level T.
 * Tl = line j, Tm = line j-1, Tp = line j+1.
 * Sm, Sl, Sp: the same three lines of the field at which lambda, c_V and X are EVALUATED.  In the
 * paper's scheme that is the current level itself (S == T: "without using iterations"); in
 * the iterated variant (orc_step_picard below) it is the previous iterate of the new level. */
static void regular_row(const orc_ctx *c, int b, int i, int j, int m, real tau, real amp,
                        const real *Tm, const real *Tl, const real *Tp,
                        const real *Sm, const real *Sl, const real *Sp,
                        real *A, real *B, real *C, real *F)
{
    const orc_layer *Lm = &c->layers[m];
    const double *r = c->r, *z = c->z;
    real h_i = (real)r[i] - (real)r[i - 1];          /* h_i = r_i - r_{i-1} */
    real h_ip = (real)r[i + 1] - (real)r[i];
    real hbar = (h_ip + h_i) / 2;                    /* hbar_i */
    real eta_j = (real)z[j] - (real)z[j - 1];        /* eta_j = z_j - z_{j-1} */
    real eta_jp = (real)z[j + 1] - (real)z[j];
    real etabar = (eta_jp + eta_j) / 2;              /* G2 */
    real r_i = (real)r[i];
    real r_mh = ((real)r[i] + (real)r[i - 1]) / 2;   /* r_{i-1/2} */
    real r_ph = ((real)r[i] + (real)r[i + 1]) / 2;   /* r_{i+1/2} */
    real T_ij = Tl[i];
    real S_ij = Sl[i];
    real lam_mh = face_lambda(c, &Lm->k, S_ij, Sl[i - 1]); /* lambda_{i-1/2,j} */
    real lam_ph = face_lambda(c, &Lm->k, S_ij, Sl[i + 1]); /* lambda_{i+1/2,j} */
    real lam_jm = face_lambda(c, &Lm->k, S_ij, Sm[i]);     /* lambda_{i,j-1/2} */
    real lam_jp = face_lambda(c, &Lm->k, S_ij, Sp[i]);     /* lambda_{i,j+1/2} */
    real rc = (real)Lm->rho * law_eval(&Lm->cp, S_ij);     /* rho_{i,j} c_V{i,j} */
    real X = 0;
    if (Lm->is_heater)                                     /* X_{i,j} = X_m(T_{i,j}), (2)-(4) */
        X = (real)c->Q0[b] * law_eval(&Lm->src_shape, S_ij) * amp;
    /* Lambda_j[T_{i,j}], eq. (11) */
    real Lj = (1 / etabar) * (lam_jp * (Tp[i] - T_ij) / eta_jp - lam_jm * (T_ij - Tm[i]) / eta_j);
    *A = -r_mh * lam_mh / (r_i * hbar * h_i);
    *B = (1 / (r_i * hbar)) * (r_mh * lam_mh / h_i + r_ph * lam_ph / h_ip) + rc / tau;
    *C = -r_ph * lam_ph / (r_i * hbar * h_ip);
    *F = rc / tau * T_ij + Lj + X;
}

/* One line j of batch member b: forward sweep (12),(16),(20), then (17) and back sweep (14).
 * N = N_j, the last node of the line (9) P:L117: nr - 1 on a rectangle; on the stepped domain (G24)
 * the lines above the step end at i_step with the zero-flux condition (6),(15), and the nodes beyond
 * N_j are not part of Omega: they keep their value. */
static void line_solve(const orc_ctx *c, int b, int j, real tau, real amp,
                       const real *T, const real *S, real *Tn, real *alpha, real *beta)
{
    int nr = c->nr;
    int shortline = (c->j_step > 0 && j > c->j_step);
    int N = shortline ? c->i_step : nr - 1;
    const real *Tm = T + (size_t)(j - 1) * nr, *Tl = T + (size_t)j * nr, *Tp = T + (size_t)(j + 1) * nr;
    const real *Sm = S + (size_t)(j - 1) * nr, *Sl = S + (size_t)j * nr, *Sp = S + (size_t)(j + 1) * nr;
    real *out = Tn + (size_t)j * nr;
    const uint8_t *seg = c->seg_layer + (size_t)b * (nr - 1);
    const double *r = c->r;

    /* (15),(16) P:L158-169: T^_0 = T^_1  <=>  alpha_0 = 1, beta_0 = 0 */
    if (c->r_in.kind == ORC_BC_NEUMANN0) {
        alpha[0] = 1;
        beta[0] = 0;
    } else {
        alpha[0] = 0;
        beta[0] = (real)c->r_in.value;
    }
    for (int i = 1; i <= N - 1; ++i) {
        int m = seg[i - 1], m1 = seg[i];
        if (m != m1) {
            /* interface node i*, eq. (20), lambda* = lambda(T_{i*,j}) P:L183 */
            real lam_m = law_eval(&c->layers[m].k, Sl[i]);
            real lam_m1 = law_eval(&c->layers[m1].k, Sl[i]);
            real h_i = (real)r[i] - (real)r[i - 1];
            real h_ip = (real)r[i + 1] - (real)r[i];
            real den = lam_m1 * h_i + lam_m * h_ip * (1 - alpha[i - 1]);
            alpha[i] = lam_m1 * h_i / den;
            beta[i] = lam_m * h_ip * beta[i - 1] / den;
        } else {
            real A, B, C, F;
            regular_row(c, b, i, j, m, tau, amp, Tm, Tl, Tp, Sm, Sl, Sp, &A, &B, &C, &F);
            /* (12) P:L133-136 */
            real den = B + A * alpha[i - 1];
            alpha[i] = -C / den;
            beta[i] = (F - A * beta[i - 1]) / den;
        }
    }
    /* (17) P:L171-174 */
    if (shortline || c->r_out.kind == ORC_BC_NEUMANN0)
        out[N] = beta[N - 1] / (1 - alpha[N - 1]);
    else
        out[N] = (real)c->r_out.value;
    for (int i = N + 1; i < nr; ++i) out[i] = Tl[i]; /* outside Omega */
    /* (14) P:L150 */
    for (int i = N - 1; i >= 0; --i)
        out[i] = alpha[i] * out[i + 1] + beta[i];
}

/* Stepped domain (G24): the face z = z_{j_step}, i > i_step carries no flux (6).  First order, like the
 * z boundaries (G16): the nodes just above it mirror the new values of the nodes below, so that the
 * explicit flux lambda (T_{i,j+1} - T_{i,j}) / eta through that face is zero in the next step. */
static void step_face(const orc_ctx *c, real *Tn)
{
    if (c->j_step <= 0) return;
    for (int i = c->i_step + 1; i < c->nr; ++i)
        Tn[(size_t)(c->j_step + 1) * c->nr + i] = Tn[(size_t)c->j_step * c->nr + i];
}

/* ------------------------------------------------------------------ life cycle */

static int validate(const orc_desc *d)
{
    if (!d || d->nr < 3 || d->nz < 3 || d->batch < 1 || d->nlayers < 1 || d->nlayers > 255) return 1;
    if (!(d->dt > 0)) return 1;
    for (int i = 1; i < d->nr; ++i)
        if (!(d->r[i] > d->r[i - 1])) return 1;
    if (d->r[0] < 0) return 1;
    for (int j = 1; j < d->nz; ++j)
        if (!(d->z[j] > d->z[j - 1])) return 1;
    for (int b = 0; b < d->batch; ++b) {
        const uint8_t *seg = d->seg_layer + (size_t)b * (d->nr - 1);
        for (int i = 0; i < d->nr - 1; ++i)
            if (seg[i] >= d->nlayers) return 1;
        for (int i = 1; i < d->nr - 2; ++i) /* two adjacent interface nodes */
            if (seg[i - 1] != seg[i] && seg[i] != seg[i + 1]) return 1;
    }
    if (d->steps_per_period < 0 || d->steps_on < 0 || d->steps_on > d->steps_per_period) return 1;
    if (d->transient_substeps < 0) return 1;
    if (d->transient_substeps > 0 && !(d->transient_k > 0)) return 1;
    if (d->nprobes < 0 || (d->nprobes > 0 && d->probe_every < 1)) return 1;
    for (int p = 0; p < d->nprobes; ++p) {
        int i = d->probe_ij[2 * p], j = d->probe_ij[2 * p + 1];
        if (i < 0 || i >= d->nr || j < 0 || j >= d->nz) return 1;
        if (d->j_step > 0 && j > d->j_step && i > d->i_step) return 1; /* outside Omega */
    }
    if (d->j_step != 0 || d->i_step != 0) {
        if (d->j_step < 1 || d->j_step > d->nz - 3) return 1;
        if (d->i_step < 2 || d->i_step > d->nr - 2) return 1;
    }
    return 0;
}

void orc_destroy(orc_ctx *c)
{
    if (!c) return;
    free(c->r); free(c->z); free(c->layers); free(c->seg_layer); free(c->Q0);
    free(c->probe_ij); free(c->T); free(c->Tn); free(c->Ts); free(c->alpha); free(c->beta); free(c->probe);
    free(c);
}

static void *dup_mem(const void *src, size_t bytes)
{
    void *p = malloc(bytes ? bytes : 1);
    if (p && src && bytes) memcpy(p, src, bytes);
    return p;
}

orc_ctx *orc_create(const orc_desc *d)
{
    if (validate(d)) return NULL;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof *c);
    if (!c) return NULL;
    c->nr = d->nr; c->nz = d->nz; c->batch = d->batch; c->nlayers = d->nlayers;
    c->r = (double *)dup_mem(d->r, sizeof(double) * d->nr);
    c->z = (double *)dup_mem(d->z, sizeof(double) * d->nz);
    c->layers = (orc_layer *)dup_mem(d->layers, sizeof(orc_layer) * d->nlayers);
    c->seg_layer = (uint8_t *)dup_mem(d->seg_layer, (size_t)d->batch * (d->nr - 1));
    c->r_in = d->r_in; c->r_out = d->r_out; c->z_lo = d->z_lo; c->z_hi = d->z_hi;
    c->dt = d->dt;
    c->Q0 = (double *)calloc(d->batch, sizeof(double));
    if (d->Q0) memcpy(c->Q0, d->Q0, sizeof(double) * d->batch);
    c->steps_per_period = d->steps_per_period; c->steps_on = d->steps_on;
    c->transient_substeps = d->transient_substeps; c->face_mode = d->face_mode;
    c->transient_k = d->transient_k;
    c->nprobes = d->nprobes; c->probe_every = d->probe_every;
    c->i_step = d->i_step; c->j_step = d->j_step;
    c->probe_ij = (int32_t *)dup_mem(d->probe_ij, sizeof(int32_t) * 2 * (size_t)d->nprobes);
    size_t cells = (size_t)d->batch * d->nz * d->nr;
    c->T = (real *)malloc(sizeof(real) * cells);
    c->Tn = (real *)malloc(sizeof(real) * cells);
    c->alpha = (real *)malloc(sizeof(real) * (size_t)d->nz * d->nr);
    c->beta = (real *)malloc(sizeof(real) * (size_t)d->nz * d->nr);
    if (!c->T || !c->Tn || !c->alpha || !c->beta) { orc_destroy(c); return NULL; }

    int nr = c->nr, nz = c->nz;
    for (int b = 0; b < c->batch; ++b) {
        real *T = c->T + (size_t)b * nz * nr;
        for (size_t k = 0; k < (size_t)nz * nr; ++k)
            T[k] = d->T_init ? (real)d->T_init[(size_t)b * nz * nr + k] : (real)d->T0; /* (5) */
        if (!d->T_init) {
            /* Dirichlet sides hold their value from t = 0 (6); r sides first, z lines last
             * so that corners belong to the z lines (G17) */
            if (c->r_in.kind == ORC_BC_DIRICHLET)
                for (int j = 0; j < nz; ++j) T[(size_t)j * nr] = (real)c->r_in.value;
            if (c->r_out.kind == ORC_BC_DIRICHLET)
                for (int j = 0; j < nz; ++j) T[(size_t)j * nr + nr - 1] = (real)c->r_out.value;
            if (c->z_lo.kind == ORC_BC_DIRICHLET)
                for (int i = 0; i < nr; ++i) T[i] = (real)c->z_lo.value;
            if (c->z_hi.kind == ORC_BC_DIRICHLET)
                for (int i = 0; i < nr; ++i) T[(size_t)(nz - 1) * nr + i] = (real)c->z_hi.value;
        }
    }
    for (int b = 0; b < c->batch; ++b) step_face(c, c->T + (size_t)b * nz * nr);
    memcpy(c->Tn, c->T, sizeof(real) * cells);
    return c;
}

static void append_probes(orc_ctx *c)
{
    int64_t rec = (int64_t)c->batch * c->nprobes;
    if (c->probe_len + rec > c->probe_cap) {
        int64_t cap = c->probe_cap ? 2 * c->probe_cap : 1024;
        while (cap < c->probe_len + rec) cap *= 2;
        c->probe = (double *)realloc(c->probe, sizeof(double) * (size_t)cap);
        c->probe_cap = cap;
    }
    for (int b = 0; b < c->batch; ++b)
        for (int p = 0; p < c->nprobes; ++p) {
            int i = c->probe_ij[2 * p], j = c->probe_ij[2 * p + 1];
            c->probe[c->probe_len++] = (double)c->T[((size_t)b * c->nz + j) * c->nr + i];
        }
}

/* n solver steps T -> T^ (a transient sub-step counts as one step). */
void orc_step(orc_ctx *c, int64_t n)
{
    int nr = c->nr, nz = c->nz, M = nz - 1;
    for (int64_t s = 0; s < n; ++s) {
        double tau_d, amp_d;
        orc_schedule(c, c->step, &tau_d, &amp_d);
        real tau = (real)tau_d, amp = (real)amp_d;
        for (int b = 0; b < c->batch; ++b) {
            const real *T = c->T + (size_t)b * nz * nr;
            real *Tn = c->Tn + (size_t)b * nz * nr;
            /* "the cycle for j-index from 1 to M-1 is parallelized" */
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
            for (int j = 1; j <= M - 1; ++j)
                line_solve(c, b, j, tau, amp, T, T, Tn, c->alpha + (size_t)j * nr, c->beta + (size_t)j * nr);
            /* z boundaries (G16, G17; "constructed in a similar way" P:L164) */
            for (int i = 0; i < nr; ++i) {
                Tn[i] = (c->z_lo.kind == ORC_BC_DIRICHLET) ? T[i] : Tn[(size_t)1 * nr + i];
                Tn[(size_t)M * nr + i] =
                    (c->z_hi.kind == ORC_BC_DIRICHLET) ? T[(size_t)M * nr + i] : Tn[(size_t)(M - 1) * nr + i];
            }
            step_face(c, Tn);
        }
        real *t = c->T; c->T = c->Tn; c->Tn = t; /* swap levels */
        c->step += 1;
        if (c->nprobes > 0 && c->step % c->probe_every == 0) append_probes(c);
    }
}

/* Variant, not the paper's scheme: "for implicit difference schema with
 * coefficients depending on the sought-after function (temperature), one needs to make iterations
 * for evaluation of temperature at each time step" -- which the paper avoids.
 * Simple (Picard) iteration on the coefficients, reading G23: T^(0) = T; T^(s+1) solves (8)-(20) with
 * every lambda, c_V and X evaluated at T^(s) instead of T, while T itself stays where (8) has the
 * current level: in rho c_V (T^ - T)/tau and in Lambda_j[T].  T^ = T^(iters); iters = 1 is orc_step. */
void orc_step_picard(orc_ctx *c, int64_t n, int iters)
{
    int nr = c->nr, nz = c->nz, M = nz - 1;
    size_t cells = (size_t)c->batch * nz * nr;
    if (iters < 1) return;
    if (!c->Ts) c->Ts = (real *)malloc(sizeof(real) * cells);
    for (int64_t s = 0; s < n; ++s) {
        double tau_d, amp_d;
        orc_schedule(c, c->step, &tau_d, &amp_d);
        real tau = (real)tau_d, amp = (real)amp_d;
        const real *S = c->T;      /* T^(0) = T */
        real *out = c->Tn;
        for (int it = 0; it < iters; ++it) {
            for (int b = 0; b < c->batch; ++b) {
                const real *T = c->T + (size_t)b * nz * nr;
                const real *Sb = S + (size_t)b * nz * nr;
                real *Tn = out + (size_t)b * nz * nr;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
                for (int j = 1; j <= M - 1; ++j)
                    line_solve(c, b, j, tau, amp, T, Sb, Tn, c->alpha + (size_t)j * nr, c->beta + (size_t)j * nr);
                /* z boundaries of the iterate, as in orc_step */
                for (int i = 0; i < nr; ++i) {
                    Tn[i] = (c->z_lo.kind == ORC_BC_DIRICHLET) ? T[i] : Tn[(size_t)1 * nr + i];
                    Tn[(size_t)M * nr + i] =
                        (c->z_hi.kind == ORC_BC_DIRICHLET) ? T[(size_t)M * nr + i] : Tn[(size_t)(M - 1) * nr + i];
                }
                step_face(c, Tn);
            }
            S = out;                                  /* the next iteration evaluates the laws here */
            out = (out == c->Tn) ? c->Ts : c->Tn;     /* ... and writes into the other buffer */
        }
        /* S is T^(iters): make it the current level */
        if (S == c->Tn) { real *t = c->T; c->T = c->Tn; c->Tn = t; }
        else { real *t = c->T; c->T = c->Ts; c->Ts = t; }
        c->step += 1;
        if (c->nprobes > 0 && c->step % c->probe_every == 0) append_probes(c);
    }
}

/* ------------------------------------------------------------------ access */

int64_t orc_step_index(const orc_ctx *c) { return c->step; }

void orc_get_field(const orc_ctx *c, int b, double *dst)
{
    size_t n = (size_t)c->nz * c->nr;
    const real *T = c->T + (size_t)b * n;
    for (size_t k = 0; k < n; ++k) dst[k] = (double)T[k];
}

void orc_set_field(orc_ctx *c, int b, const double *src, int64_t step_index)
{
    size_t n = (size_t)c->nz * c->nr;
    real *T = c->T + (size_t)b * n;
    for (size_t k = 0; k < n; ++k) T[k] = (real)src[k];
    step_face(c, T);
    c->step = step_index;
}

int64_t orc_probe(const orc_ctx *c, double *dst, int64_t max)
{
    int64_t n = c->probe_len < max ? c->probe_len : max;
    if (dst && n > 0) memcpy(dst, c->probe, sizeof(double) * (size_t)n);
    return c->probe_len;
}

/* The rows of line j of batch member b as the next orc_step would see them, one tridiagonal
 * row A_i x_{i-1} + B_i x_i + C_i x_{i+1} = F_i per node i = 0..N: (15) at the r boundaries,
 * (13) at regular nodes, the flux-continuity relation (18) P:L178-181 (new level, G7) at
 * interface nodes.  Used by the dense-solve pin: the sweep above never reads these arrays. */
void orc_line_rows(const orc_ctx *c, int b, int j, double *A, double *B, double *C, double *F)
{
    int nr = c->nr, nz = c->nz;
    int shortline = (c->j_step > 0 && j > c->j_step);
    int N = shortline ? c->i_step : nr - 1;
    double tau_d, amp_d;
    orc_schedule(c, c->step, &tau_d, &amp_d);
    const real *T = c->T + (size_t)b * nz * nr;
    const real *Tm = T + (size_t)(j - 1) * nr, *Tl = T + (size_t)j * nr, *Tp = T + (size_t)(j + 1) * nr;
    const uint8_t *seg = c->seg_layer + (size_t)b * (nr - 1);
    if (c->r_in.kind == ORC_BC_NEUMANN0) { A[0] = 0; B[0] = 1; C[0] = -1; F[0] = 0; }
    else { A[0] = 0; B[0] = 1; C[0] = 0; F[0] = c->r_in.value; }
    if (shortline || c->r_out.kind == ORC_BC_NEUMANN0) { A[N] = -1; B[N] = 1; C[N] = 0; F[N] = 0; }
    else { A[N] = 0; B[N] = 1; C[N] = 0; F[N] = c->r_out.value; }
    for (int i = N + 1; i < nr; ++i) { A[i] = 0; B[i] = 1; C[i] = 0; F[i] = (double)Tl[i]; } /* outside Omega */
    for (int i = 1; i <= N - 1; ++i) {
        int m = seg[i - 1], m1 = seg[i];
        if (m != m1) {
            real lam_m = law_eval(&c->layers[m].k, Tl[i]);
            real lam_m1 = law_eval(&c->layers[m1].k, Tl[i]);
            real h_i = (real)c->r[i] - (real)c->r[i - 1];
            real h_ip = (real)c->r[i + 1] - (real)c->r[i];
            A[i] = (double)(-lam_m / h_i);
            B[i] = (double)(lam_m / h_i + lam_m1 / h_ip);
            C[i] = (double)(-lam_m1 / h_ip);
            F[i] = 0;
        } else {
            real a, bb, cc, f;
            regular_row(c, b, i, j, m, (real)tau_d, (real)amp_d, Tm, Tl, Tp, Tm, Tl, Tp, &a, &bb, &cc, &f);
            A[i] = (double)a; B[i] = (double)bb; C[i] = (double)cc; F[i] = (double)f;
        }
    }
}

/* Stability bound (21) P:L194-196: tau <= (min eta_j^2 / 2) * min rho c_V / lambda, the second
 * minimum over layers and over T on [T_lo, T_hi] sampled at nsamp equidistant points (G19). */
double orc_stable_dt(const orc_desc *d, double T_lo, double T_hi, int nsamp)
{
    double eta2 = INFINITY, ratio = INFINITY;
    for (int j = 1; j < d->nz; ++j) {
        double e = d->z[j] - d->z[j - 1];
        if (e * e < eta2) eta2 = e * e;
    }
    if (nsamp < 2) nsamp = 2;
    for (int m = 0; m < d->nlayers; ++m)
        for (int s = 0; s < nsamp; ++s) {
            double T = T_lo + (T_hi - T_lo) * (double)s / (double)(nsamp - 1);
            double q = fabs(d->layers[m].rho * (double)law_eval(&d->layers[m].cp, (real)T) /
                            (double)law_eval(&d->layers[m].k, (real)T)); /* |rho c_V / lambda| */
            if (q < ratio) ratio = q;
        }
    return eta2 / 2 * ratio;
}

double orc_law_eval(const orc_law *L, double T) { return (double)law_eval(L, (real)T); }

int orc_real_bytes(void) { return (int)sizeof(real); }

int orc_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
