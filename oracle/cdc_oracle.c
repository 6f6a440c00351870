/*
 * cdc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU statement of what the seed scan of
 * arXiv 1908.01949 computes (PAPER.md = /root/reference/PAPER.md at build time).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code with
 * paper_1908_01949_b200/csrc/ and neither includes the other.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py).
 * -ffp-contract=off matters: with +,-,*,/,sqrt only and no fused multiply-add
 * the results are IEEE-754 reproducible, which is what lets the GPU's fp64
 * re-score (A8/A9) be compared bit for bit.
 *
 * What follows the paper and what is a reading of it (DESIGN.md lists every reading):
 *   seed (theta, z, px, py, pz) at R0 = 50 cm ............ PAPER.md:51 (sec. 2.1)
 *   RKN propagation of the track ......................... PAPER.md:55 (sec. 2.2, ref [5]);
 *       the stage formula is not printed -> textbook 4th-order Nystroem scheme (reading C5)
 *   DCA between the extrapolated track and a fired wire .. PAPER.md:55; located on the stepped
 *       track by the sign change of d(dist^2)/ds, chord interpolation (reading C9)
 *   E = sum_wires min(d_L^2, d_R^2, lambda) ............... PAPER.md:65-69, Eq. (1);
 *       d_L, d_R = D -+ drift, so min(d_L^2, d_R^2) = (D - drift)^2; S = sum (1 - d^2/lambda) over
 *       matched terms, E = lambda (N_terms - S) (reading C10)
 *   "hits with d^2 < lambda are classified" .............. PAPER.md:69 -> labels (reading C12)
 *   Hough circle finding -> (theta0, px0, py0) ranges .... PAPER.md:51, :61 (Fig. 4); parametrisation
 *       unstated -> (cx, cy, R) accumulator, gather form (reading C13)
 *
 * Pins (tests/test_oracle_pins.py, none of them re-derives the oracle from itself):
 *   RKN: analytic helix < 1e-6 mm after 3 turns, T_z bit-constant, |T| drift, 4th-order ratio 16
 *   field: closed forms of the tabulated B_r/B_z, zero discrete divergence
 *   geometry: wire counts, end-plate radii/azimuth closed forms
 *   lookup: exhaustive scan over all hit wires x all intervals gives the identical triples
 *   D: skew-line closed form, dense helix resampling within the sagitta bound
 *   score: E = lambda (N - S); 0 <= S <= n_match; truth node maximal on a smear-free event
 *   energy loss: p_final = p0 - eps h m exactly; eps = 0 reduces to the plain scheme
 *   Hough: noise-free exact circle -> peak bin holds the true (c, R), count = number of hits
 * Parity unpinned: the paper's own efficiency/purity figures (need COMET MC) -- not computed here.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_KAPPA 0.299792458 /* curvature[1/mm] = kappa q B[T] / p[MeV/c]  (reading C1) */

typedef struct {
    int32_t n_layers;
    const double *r_mm;       /* waist radius of layer j (radius at z = 0) */
    const int32_t *n_wires;   /* wires in layer j */
    const double *phi0;       /* azimuth of wire 0 of layer j at z = 0 */
    const double *stereo;     /* signed stereo angle of layer j */
    const int32_t *offset;    /* n_layers + 1 prefix sums */
    int32_t n_wires_total;
    const float *wire;        /* [W][5] = w0x, w0y, ux, uy, uz  (canonical fp32 input) */
    double z_half, R0, r_out;
} orc_geom;

typedef struct {
    int32_t kind;             /* 0 uniform (0,0,bz); 1 (r,z) table, bilinear */
    double bz;
    int32_t nr, nz;
    double r0, z0, dr, dz;
    const float *tab;         /* [nz][nr][2] = B_r, B_z  (canonical fp32 input) */
} orc_field;

typedef struct {
    double h;                 /* fixed step, mm */
    int32_t max_steps;
    double window;            /* match iff (D - drift)^2 < window^2 */
    double eloss;             /* MeV per mm of in-gas path */
    int32_t charge;           /* -1 for e- */
} orc_params;

typedef struct {
    int32_t n_hits;
    const int32_t *wire_id;   /* ascending, distinct */
    const float *drift;       /* mm */
} orc_hits;

typedef struct {              /* one owned approach to a hit wire */
    int32_t interval, hit, wire, turn, matched;
    double D, resid, zw;
} orc_approach;

typedef struct {
    int32_t n_match, n_steps, turns, m_gas;
    double chi2;
    double r[3], T[3], p;
    int32_t n_rec;            /* approach records written (<= cap) */
} orc_result;

/* ---- C3: field ---------------------------------------------------------- */
void orc_field_at(const orc_field *f, double x, double y, double z, double *B)
{
    if (f->kind == 0) { B[0] = 0.0; B[1] = 0.0; B[2] = f->bz; return; }
    double rho = sqrt(x * x + y * y);
    double fr = (rho - f->r0) / f->dr;
    double fz = (z - f->z0) / f->dz;
    int ir = (int)floor(fr), iz = (int)floor(fz);
    if (ir < 0) ir = 0;
    if (ir > f->nr - 2) ir = f->nr - 2;
    if (iz < 0) iz = 0;
    if (iz > f->nz - 2) iz = f->nz - 2;
    double wr = fr - (double)ir, wz = fz - (double)iz;
    const float *n00 = f->tab + ((size_t)iz * f->nr + ir) * 2;
    const float *n01 = n00 + 2;
    const float *n10 = n00 + (size_t)f->nr * 2;
    const float *n11 = n10 + 2;
    double Br = (1.0 - wz) * ((1.0 - wr) * (double)n00[0] + wr * (double)n01[0])
              + wz * ((1.0 - wr) * (double)n10[0] + wr * (double)n11[0]);
    double Bz = (1.0 - wz) * ((1.0 - wr) * (double)n00[1] + wr * (double)n01[1])
              + wz * ((1.0 - wr) * (double)n10[1] + wr * (double)n11[1]);
    if (rho > 0.0) { B[0] = Br * x / rho; B[1] = Br * y / rho; }
    else           { B[0] = 0.0; B[1] = 0.0; }
    B[2] = Bz;
}

/* ---- C5: one Nystroem-RK4 step of r'' = a (r' x B(r)) ------------------- */
static void cross_scaled(double a, const double *T, const double *B, double *k)
{
    k[0] = a * (T[1] * B[2] - T[2] * B[1]);
    k[1] = a * (T[2] * B[0] - T[0] * B[2]);
    k[2] = a * (T[0] * B[1] - T[1] * B[0]);
}

void orc_rkn_step(const orc_field *f, double a, double h, const double *r, const double *T,
                  double *rn, double *Tn)
{
    double B[3], k1[3], k2[3], k3[3], k4[3], q[3], U[3];
    int i;
    orc_field_at(f, r[0], r[1], r[2], B);
    cross_scaled(a, T, B, k1);
    for (i = 0; i < 3; ++i) q[i] = r[i] + (h / 2.0) * T[i] + (h * h / 8.0) * k1[i];
    orc_field_at(f, q[0], q[1], q[2], B);
    for (i = 0; i < 3; ++i) U[i] = T[i] + (h / 2.0) * k1[i];
    cross_scaled(a, U, B, k2);
    for (i = 0; i < 3; ++i) U[i] = T[i] + (h / 2.0) * k2[i];
    cross_scaled(a, U, B, k3);
    for (i = 0; i < 3; ++i) q[i] = r[i] + h * T[i] + (h * h / 2.0) * k3[i];
    orc_field_at(f, q[0], q[1], q[2], B);
    for (i = 0; i < 3; ++i) U[i] = T[i] + h * k3[i];
    cross_scaled(a, U, B, k4);
    for (i = 0; i < 3; ++i) {
        rn[i] = r[i] + h * T[i] + (h * h / 6.0) * (k1[i] + k2[i] + k3[i]);
        Tn[i] = T[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    }
}

/* The same step, plus the local error estimate of the adaptive Runge-Kutta-Nystroem propagator of PAPER.md ref. [5]
 * (Lund et al., JINST 4 P04001): err = h^2 max_i |k1_i - k2_i - k3_i + k4_i|, each component
 * evaluated left to right (reading C19).  rn, Tn are bit-equal to orc_rkn_step's. */
void orc_rkn_step_err(const orc_field *f, double a, double h, const double *r, const double *T,
                      double *rn, double *Tn, double *err)
{
    double B[3], k1[3], k2[3], k3[3], k4[3], q[3], U[3];
    double emax = 0.0;
    int i;
    orc_field_at(f, r[0], r[1], r[2], B);
    cross_scaled(a, T, B, k1);
    for (i = 0; i < 3; ++i) q[i] = r[i] + (h / 2.0) * T[i] + (h * h / 8.0) * k1[i];
    orc_field_at(f, q[0], q[1], q[2], B);
    for (i = 0; i < 3; ++i) U[i] = T[i] + (h / 2.0) * k1[i];
    cross_scaled(a, U, B, k2);
    for (i = 0; i < 3; ++i) U[i] = T[i] + (h / 2.0) * k2[i];
    cross_scaled(a, U, B, k3);
    for (i = 0; i < 3; ++i) q[i] = r[i] + h * T[i] + (h * h / 2.0) * k3[i];
    orc_field_at(f, q[0], q[1], q[2], B);
    for (i = 0; i < 3; ++i) U[i] = T[i] + h * k3[i];
    cross_scaled(a, U, B, k4);
    for (i = 0; i < 3; ++i) {
        double e = k1[i] - k2[i] - k3[i] + k4[i];
        rn[i] = r[i] + h * T[i] + (h * h / 6.0) * (k1[i] + k2[i] + k3[i]);
        Tn[i] = T[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
        if (fabs(e) > emax) emax = fabs(e);
    }
    *err = h * h * emax;
}

/* ---- C9: offset of a point from a wire line, and g = delta . T ---------- */
static void wire_delta(const float *w, const double *r, double *delta, double *tpar)
{
    double dx = r[0] - (double)w[0], dy = r[1] - (double)w[1], dz = r[2];
    double ux = (double)w[2], uy = (double)w[3], uz = (double)w[4];
    double t = dx * ux + dy * uy + dz * uz;
    delta[0] = dx - t * ux;
    delta[1] = dy - t * uy;
    delta[2] = dz - t * uz;
    *tpar = t;
}

static double wire_g(const float *w, const double *r, const double *T)
{
    double d[3], t;
    wire_delta(w, r, d, &t);
    return d[0] * T[0] + d[1] * T[1] + d[2] * T[2];
}

/* ---- C8: candidate wires near r (acceleration only; superset) ----------- */
static int lookup_candidates(const orc_geom *g, const double *r, int32_t *cand /* >= 5 per layer in reach */,
                             int cand_cap)
{
    int n = 0, j, dk;
    double rho2 = r[0] * r[0] + r[1] * r[1];
    double phi = atan2(r[1], r[0]);
    double pitch = 1e300;
    for (j = 1; j < g->n_layers; ++j)
        if (g->r_mm[j] - g->r_mm[j - 1] < pitch) pitch = g->r_mm[j] - g->r_mm[j - 1];
    for (j = 0; j < g->n_layers; ++j) {
        double te = tan(g->stereo[j]);
        double u2 = rho2 - r[2] * r[2] * te * te;        /* hyperboloid coordinate: u = r_j on the layer */
        double u = sqrt(u2 > 0.0 ? u2 : 0.0);
        if (fabs(u - g->r_mm[j]) > 1.5 * pitch) continue; /* the three nearest layers */
        int nj = g->n_wires[j];
        double sh = atan(r[2] * te / g->r_mm[j]);         /* stereo shift of the azimuth at height z */
        double kf = (phi - g->phi0[j] - sh) * (double)nj / (2.0 * M_PI);
        long kc = (long)floor(kf + 0.5);
        for (dk = -2; dk <= 2 && n < cand_cap; ++dk) {
            long k = (kc + dk) % nj;
            if (k < 0) k += nj;
            cand[n++] = g->offset[j] + (int32_t)k;
        }
    }
    /* ascending wire id so that the summation order equals the exhaustive scan's */
    for (j = 1; j < n; ++j) {
        int32_t v = cand[j];
        int i = j - 1;
        while (i >= 0 && cand[i] > v) { cand[i + 1] = cand[i]; --i; }
        cand[i + 1] = v;
    }
    return n;
}

/* ---- C4-C10: evaluate one seed ------------------------------------------
 * mode 0: exhaustive (every hit wire tested in every in-gas interval) -- the plain definition
 * mode 1: layer/cell lookup (layers within 1.5 pitches x 5 cells) -- must give identical results (pinned)
 * hit_of_wire: dense table, hit index or -1.  rec/rec_cap: optional approach records, kept when
 * D < drift + window + rec_slack.  traj (optional): (max_steps+1) x 6 vertices (r, T). */
void orc_eval_seed(const orc_geom *g, const orc_field *f, const orc_hits *hits,
                   const int32_t *hit_of_wire, const double *seed, const orc_params *P, int32_t mode,
                   orc_result *out, orc_approach *rec, int32_t rec_cap, double rec_slack, double *traj)
{
    double r[3], T[3], rn[3], Tn[3];
    double lambda = P->window * P->window;
    double p0, p;
    int32_t n = 0, t = 0, m = 0, n_match = 0, n_rec = 0;
    double chi2 = 0.0;
    int c_n = 1, c_next;
    int32_t cand[32];
    int i;

    /* C4: seed -> state */
    r[0] = g->R0 * cos(seed[0]);
    r[1] = g->R0 * sin(seed[0]);
    r[2] = seed[1];
    p0 = sqrt(seed[2] * seed[2] + seed[3] * seed[3] + seed[4] * seed[4]);
    T[0] = seed[2] / p0; T[1] = seed[3] / p0; T[2] = seed[4] / p0;
    p = p0;
    if (traj) { memcpy(traj, r, 24); memcpy(traj + 3, T, 24); }

    while (n < P->max_steps) {
        double a = (ORC_KAPPA * (double)P->charge) / p;
        orc_rkn_step(f, a, P->h, r, T, rn, Tn);
        /* C8/C9: score interval n (only if its start vertex is in the gas) */
        if (c_n) {
            int nc, ic;
            if (mode == 0) nc = hits->n_hits;
            else nc = lookup_candidates(g, r, cand, 32);
            for (ic = 0; ic < nc; ++ic) {
                int32_t hidx, wid;
                if (mode == 0) { hidx = ic; wid = hits->wire_id[ic]; }
                else { wid = cand[ic]; hidx = hit_of_wire[wid]; if (hidx < 0) continue; }
                const float *w = g->wire + (size_t)wid * 5;
                double g0 = wire_g(w, r, T);
                if (!(g0 <= 0.0)) continue;
                double g1 = wire_g(w, rn, Tn);
                if (!(g1 > 0.0)) continue;
                double tau = g0 / (g0 - g1);
                double Pp[3], d[3], tpar;
                for (i = 0; i < 3; ++i) Pp[i] = r[i] + tau * (rn[i] - r[i]);
                wire_delta(w, Pp, d, &tpar);
                double D = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                double zw = tpar * (double)w[4];
                double x = (double)hits->drift[hidx];
                double resid = D - x;
                int inside = fabs(zw) <= g->z_half;
                int matched = inside && (resid * resid < lambda);
                if (matched) { n_match += 1; chi2 += resid * resid; }
                if (rec && n_rec < rec_cap && D < x + P->window + rec_slack) {
                    orc_approach *q = rec + n_rec++;
                    q->interval = n; q->hit = hidx; q->wire = wid; q->turn = t; q->matched = matched;
                    q->D = D; q->resid = resid; q->zw = zw;
                }
            }
            m += 1;                                   /* C6: one more in-gas step */
        }
        /* advance */
        for (i = 0; i < 3; ++i) { r[i] = rn[i]; T[i] = Tn[i]; }
        n += 1;
        p = p0 - (P->eloss * P->h) * (double)m;       /* C6 */
        c_next = (r[0] * r[0] + r[1] * r[1] >= g->R0 * g->R0);
        if (!c_n && c_next) t += 1;                   /* C7: turn counter */
        c_n = c_next;
        if (traj) { memcpy(traj + 6 * (size_t)n, r, 24); memcpy(traj + 6 * (size_t)n + 3, T, 24); }
        /* C7: termination */
        if (fabs(r[2]) > g->z_half) break;
        if (r[0] * r[0] + r[1] * r[1] > g->r_out * g->r_out) break;
        if (!(p > 1.0)) break;
        if (!(isfinite(r[0]) && isfinite(r[1]) && isfinite(r[2]) &&
              isfinite(T[0]) && isfinite(T[1]) && isfinite(T[2]))) break;
    }
    out->n_match = n_match; out->chi2 = chi2; out->n_steps = n; out->turns = t; out->m_gas = m;
    for (i = 0; i < 3; ++i) { out->r[i] = r[i]; out->T[i] = T[i]; }
    out->p = p; out->n_rec = n_rec;
}

void orc_seed_of_index(const double *lo, const double *step, const int32_t *nn, int64_t idx, double *seed);

/* ---- The same evaluation with the ADAPTIVE step of the propagator the paper cites ("the RKN method was
 * used for the track parameter propagation [5]"; [5] = Lund et al.) -- reading C19 applied to the scan
 * (SURVEY 8(f) #4).  Step lengths are h 2^j, j = 0..J with h 2^J <= h_max.  A trial step of length h 2^j has the error
 * estimate err = (h 2^j)^2 max_i |k1 - k2 - k3 + k4|_i (orc_rkn_step_err); if err > tol and j > 0 the trial is repeated
 * with j - 1; otherwise it is accepted, and after an accepted step with err <= tol / 32 the next trial starts one level
 * up (the estimate grows ~16-fold per doubling).  Path is counted in units of h: the step cap max_steps is a PATH cap
 * (a trial that would exceed it drops to the level that fits), the in-gas count m sums the units of the steps that
 * start in the gas, and p = p0 - eps h m (reading C6 generalised).  Everything else -- ownership of an approach by the
 * sign change of g over the (now longer) interval, chord interpolation, window, turn counter, termination -- is C7-C10
 * unchanged; the candidate wires are ALL hit wires (mode 0: the plain definition).
 * Outputs beyond orc_result: units (path in units of h), n_level[j] accepted steps per level (j < 8), and the decision
 * margins min |err - tol| / tol over rejections / acceptances and min |err - tol/32| / (tol/32) over the doubling
 * decisions (a GPU that takes its decisions in fp32 can differ where these are ~ 1e-5), and the same two distances
 * in units of the stage derivatives, min |err - threshold| / H^2 (1/mm): the estimate is H^2 times a difference of
 * four k, so the rounding noise of an fp32 evaluation is absolute in these units.  Diagnostics only: nothing of the
 * propagation or of the decisions reads them. */
typedef struct {
    int32_t units, n_level[8];
    double margin_tol, margin_up;
    uint32_t seq_hash;        /* hash of the accepted level sequence: hash = hash * 31 + (j + 1), mod 2^32 */
    double kmargin_tol, kmargin_up;
    double r0_margin;         /* min | |r_n|_xy - R0 | over the vertices n >= 1 (mm): the in-gas flag of a vertex this close to
                               * R0 is a threshold decision (diagnostic, like the margins) */
    double exit_margin;       /* min over the vertices n >= 1 of min(| |z_n| - z_half |, | |r_n|_xy - r_out |) (mm): likewise
                               * for the termination tests */
} orc_adaptive_info;

void orc_eval_seed_adaptive(const orc_geom *g, const orc_field *f, const orc_hits *hits, const double *seed,
                            const orc_params *P, double tol, double h_max, orc_result *out, orc_adaptive_info *info,
                            orc_approach *rec, int32_t rec_cap, double rec_slack)
{
    double r[3], T[3], rn[3], Tn[3];
    double lambda = P->window * P->window;
    double p0, p, err;
    int32_t n = 0, t = 0, m = 0, n_match = 0, n_rec = 0, units = 0, j = 0, J = 0, ic;
    double chi2 = 0.0;
    int c_n = 1, c_next, i;
    while (J < 7 && P->h * (double)(2 << J) <= h_max) ++J;      /* h 2^(J+1) <= h_max -> J + 1 */
    for (i = 0; i < 8; ++i) info->n_level[i] = 0;
    info->margin_tol = 1e300; info->margin_up = 1e300; info->seq_hash = 0u;
    info->kmargin_tol = 1e300; info->kmargin_up = 1e300; info->r0_margin = 1e300; info->exit_margin = 1e300;
    r[0] = g->R0 * cos(seed[0]); r[1] = g->R0 * sin(seed[0]); r[2] = seed[1];
    p0 = sqrt(seed[2] * seed[2] + seed[3] * seed[3] + seed[4] * seed[4]);
    T[0] = seed[2] / p0; T[1] = seed[3] / p0; T[2] = seed[4] / p0;
    p = p0;
    while (units < P->max_steps) {
        double a = (ORC_KAPPA * (double)P->charge) / p;
        double hj, mt;
        while (j > 0 && units + (1 << j) > P->max_steps) --j;          /* the path cap */
        for (;;) {
            hj = P->h * (double)(1 << j);
            orc_rkn_step_err(f, a, hj, r, T, rn, Tn, &err);
            mt = fabs(err - tol) / tol;
            if (mt < info->margin_tol) info->margin_tol = mt;
            if (fabs(err - tol) / (hj * hj) < info->kmargin_tol) info->kmargin_tol = fabs(err - tol) / (hj * hj);
            if (err > tol && j > 0) { --j; continue; }
            break;
        }
        if (c_n) {
            for (ic = 0; ic < hits->n_hits; ++ic) {
                const float *w = g->wire + (size_t)hits->wire_id[ic] * 5;
                double g0 = wire_g(w, r, T), g1, tau, Pp[3], d[3], tpar, D, zw, x, resid;
                int inside, matched;
                if (!(g0 <= 0.0)) continue;
                g1 = wire_g(w, rn, Tn);
                if (!(g1 > 0.0)) continue;
                tau = g0 / (g0 - g1);
                for (i = 0; i < 3; ++i) Pp[i] = r[i] + tau * (rn[i] - r[i]);
                wire_delta(w, Pp, d, &tpar);
                D = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                zw = tpar * (double)w[4];
                x = (double)hits->drift[ic];
                resid = D - x;
                inside = fabs(zw) <= g->z_half;
                matched = inside && (resid * resid < lambda);
                if (matched) { n_match += 1; chi2 += resid * resid; }
                if (rec && n_rec < rec_cap && D < x + P->window + rec_slack) {
                    orc_approach *q = rec + n_rec++;
                    q->interval = n; q->hit = ic; q->wire = hits->wire_id[ic]; q->turn = t; q->matched = matched;
                    q->D = D; q->resid = resid; q->zw = zw;
                }
            }
            m += 1 << j;
        }
        for (i = 0; i < 3; ++i) { r[i] = rn[i]; T[i] = Tn[i]; }
        n += 1; units += 1 << j; info->n_level[j] += 1; info->seq_hash = info->seq_hash * 31u + (uint32_t)(j + 1);
        p = p0 - (P->eloss * P->h) * (double)m;
        c_next = (r[0] * r[0] + r[1] * r[1] >= g->R0 * g->R0);
        if (fabs(sqrt(r[0] * r[0] + r[1] * r[1]) - g->R0) < info->r0_margin)
            info->r0_margin = fabs(sqrt(r[0] * r[0] + r[1] * r[1]) - g->R0);
        if (fabs(fabs(r[2]) - g->z_half) < info->exit_margin) info->exit_margin = fabs(fabs(r[2]) - g->z_half);
        if (fabs(sqrt(r[0] * r[0] + r[1] * r[1]) - g->r_out) < info->exit_margin)
            info->exit_margin = fabs(sqrt(r[0] * r[0] + r[1] * r[1]) - g->r_out);
        if (!c_n && c_next) t += 1;
        c_n = c_next;
        if (fabs(r[2]) > g->z_half) break;
        if (r[0] * r[0] + r[1] * r[1] > g->r_out * g->r_out) break;
        if (!(p > 1.0)) break;
        if (!(isfinite(r[0]) && isfinite(r[1]) && isfinite(r[2]) &&
              isfinite(T[0]) && isfinite(T[1]) && isfinite(T[2]))) break;
        if (j < J) {
            double mu = fabs(err - tol / 32.0) / (tol / 32.0);
            if (mu < info->margin_up) info->margin_up = mu;
            if (fabs(err - tol / 32.0) / (hj * hj) < info->kmargin_up) info->kmargin_up = fabs(err - tol / 32.0) / (hj * hj);
            if (err <= tol / 32.0) ++j;
        }
    }
    out->n_match = n_match; out->chi2 = chi2; out->n_steps = n; out->turns = t; out->m_gas = m;
    for (i = 0; i < 3; ++i) { out->r[i] = r[i]; out->T[i] = T[i]; }
    out->p = p; out->n_rec = n_rec;
    info->units = units;
}

/* exhaustive adaptive-step evaluation of a list of seeds (or of seeds [begin, end) of the grid) */
void orc_scan_adaptive(const orc_geom *g, const orc_field *f, const orc_hits *hits,
                       const double *lo, const double *step, const int32_t *nn, const int64_t *index_list,
                       int64_t begin, int64_t end, const orc_params *P, double tol, double h_max,
                       int32_t *n_match, double *chi2, int32_t *n_steps, int32_t *units, int32_t *m_gas, double *final_r,
                       int32_t *n_level /* [..][8] */, double *margins /* [..][6] */, uint32_t *seq_hash)
{
    int64_t s;
    int i;
    for (s = begin; s < end; ++s) {
        double seed[5];
        orc_result res;
        orc_adaptive_info info;
        int64_t idx = index_list ? index_list[s] : s;
        int64_t o = s - begin;
        orc_seed_of_index(lo, step, nn, idx, seed);
        orc_eval_seed_adaptive(g, f, hits, seed, P, tol, h_max, &res, &info, NULL, 0, 0.0);
        n_match[o] = res.n_match; chi2[o] = res.chi2; n_steps[o] = res.n_steps; units[o] = info.units; m_gas[o] = res.m_gas;
        final_r[3 * o] = res.r[0]; final_r[3 * o + 1] = res.r[1]; final_r[3 * o + 2] = res.r[2];
        for (i = 0; i < 8; ++i) n_level[8 * o + i] = info.n_level[i];
        margins[6 * o] = info.margin_tol; margins[6 * o + 1] = info.margin_up; seq_hash[o] = info.seq_hash;
        margins[6 * o + 2] = info.kmargin_tol; margins[6 * o + 3] = info.kmargin_up; margins[6 * o + 4] = info.r0_margin;
        margins[6 * o + 5] = info.exit_margin;
    }
}

/* seed linear index -> 5 values; axes theta, z, px, py, pz; pz fastest (tie-break order) */
void orc_seed_of_index(const double *lo, const double *step, const int32_t *nn, int64_t idx, double *seed)
{
    int a;
    for (a = 4; a >= 0; --a) {
        int64_t i = idx % nn[a];
        idx /= nn[a];
        seed[a] = lo[a] + (double)i * step[a];
    }
}

/* ---- exhaustive evaluation of seeds [begin, end) of a grid, or of a list of indices ---- */
void orc_scan(const orc_geom *g, const orc_field *f, const orc_hits *hits,
              const double *lo, const double *step, const int32_t *nn,
              const int64_t *index_list /* or NULL */, int64_t begin, int64_t end,
              const orc_params *P, int32_t mode,
              int32_t *n_match, double *chi2, int32_t *n_steps, int32_t *turns, double *final_r /* [..][3] */,
              int32_t *m_gas /* or NULL: in-gas steps (reading C6) */)
{
    int32_t *how = (int32_t *)malloc(sizeof(int32_t) * (size_t)g->n_wires_total);
    int64_t s;
    int i;
    for (i = 0; i < g->n_wires_total; ++i) how[i] = -1;
    for (i = 0; i < hits->n_hits; ++i) how[hits->wire_id[i]] = i;
    for (s = begin; s < end; ++s) {
        double seed[5];
        orc_result res;
        int64_t idx = index_list ? index_list[s] : s;
        orc_seed_of_index(lo, step, nn, idx, seed);
        orc_eval_seed(g, f, hits, how, seed, P, mode, &res, NULL, 0, 0.0, NULL);
        int64_t o = s - begin;
        n_match[o] = res.n_match; chi2[o] = res.chi2;
        if (n_steps) n_steps[o] = res.n_steps;
        if (turns) turns[o] = res.turns;
        if (m_gas) m_gas[o] = res.m_gas;
        if (final_r) { final_r[3 * o] = res.r[0]; final_r[3 * o + 1] = res.r[1]; final_r[3 * o + 2] = res.r[2]; }
    }
    free(how);
}

/* ---- C10: best seed = max S = n_match - chi2/lambda, ties -> lowest index ---- */
int64_t orc_argmax(int64_t n, const int32_t *n_match, const double *chi2, double window, double *S_best)
{
    double lambda = window * window;
    int64_t best = -1, s;
    double Sb = -1.0;
    for (s = 0; s < n; ++s) {
        double S = (double)n_match[s] - chi2[s] / lambda;
        if (S > Sb) { Sb = S; best = s; }
    }
    if (S_best) *S_best = Sb;
    return best;
}

/* ---- C12: hit -> turn labels of one seed ---------------------------------
 * label[h] = turn of the matched approach with the smallest |resid| (ties -> earliest), else -1 */
void orc_labels(const orc_geom *g, const orc_field *f, const orc_hits *hits, const double *seed,
                const orc_params *P, int32_t mode, int32_t *labels, orc_result *res_out)
{
    int32_t *how = (int32_t *)malloc(sizeof(int32_t) * (size_t)g->n_wires_total);
    int32_t cap = 16 * hits->n_hits + 1024;
    orc_approach *rec = (orc_approach *)malloc(sizeof(orc_approach) * (size_t)cap);
    double *best = (double *)malloc(sizeof(double) * (size_t)(hits->n_hits > 0 ? hits->n_hits : 1));
    orc_result res;
    int i;
    for (i = 0; i < g->n_wires_total; ++i) how[i] = -1;
    for (i = 0; i < hits->n_hits; ++i) { how[hits->wire_id[i]] = i; labels[i] = -1; best[i] = 0.0; }
    orc_eval_seed(g, f, hits, how, seed, P, mode, &res, rec, cap, 0.0, NULL);
    for (i = 0; i < res.n_rec; ++i) {
        if (!rec[i].matched) continue;
        int h = rec[i].hit;
        double ad = fabs(rec[i].resid);
        if (labels[h] < 0 || ad < best[h]) { labels[h] = rec[i].turn; best[h] = ad; }
    }
    if (res_out) *res_out = res;
    free(best); free(rec); free(how);
}

/* ---- C13: Hough circle vote, gather form ---------------------------------- */
typedef struct {
    double bin_xy, bin_R, tol, R_lo, R_hi, half_xy, origin, half_theta, half_pt;
} orc_hough_params;

void orc_hough_dims(const orc_hough_params *H, int32_t *dims /* nR, ncy, ncx */)
{
    dims[0] = (int32_t)floor((H->R_hi - H->R_lo) / H->bin_R + 0.5);
    dims[1] = (int32_t)floor(2.0 * H->half_xy / H->bin_xy + 0.5);
    dims[2] = dims[1];
}

/* accum: [nR][ncy][ncx] u32 (may be NULL); peak = (iR, icy, icx, votes); ranges[3][2] for theta0, px0, py0 */
void orc_hough(const orc_geom *g, const orc_hits *hits, double zref, const orc_hough_params *H,
               double bz, int32_t charge, uint32_t *accum, int32_t *peak, double *ranges)
{
    int32_t dims[3];
    int iR, icy, icx, h;
    orc_hough_dims(H, dims);
    double *xh = (double *)malloc(sizeof(double) * (size_t)(hits->n_hits + 1));
    double *yh = (double *)malloc(sizeof(double) * (size_t)(hits->n_hits + 1));
    for (h = 0; h < hits->n_hits; ++h) {     /* wire (x, y) at z = zref */
        const float *w = g->wire + (size_t)hits->wire_id[h] * 5;
        double t = zref / (double)w[4];
        xh[h] = (double)w[0] + t * (double)w[2];
        yh[h] = (double)w[1] + t * (double)w[3];
    }
    int64_t best_lin = -1;
    uint32_t best_votes = 0;
    int bR = 0, bcy = 0, bcx = 0;
    for (iR = 0; iR < dims[0]; ++iR) {
        double R = H->R_lo + ((double)iR + 0.5) * H->bin_R;
        for (icy = 0; icy < dims[1]; ++icy) {
            double cy = -H->half_xy + ((double)icy + 0.5) * H->bin_xy;
            for (icx = 0; icx < dims[2]; ++icx) {
                double cx = -H->half_xy + ((double)icx + 0.5) * H->bin_xy;
                int64_t lin = ((int64_t)iR * dims[1] + icy) * dims[2] + icx;
                uint32_t votes = 0;
                double cn = sqrt(cx * cx + cy * cy);
                if (fabs(cn - R) <= H->origin + H->tol) {
                    for (h = 0; h < hits->n_hits; ++h) {
                        double ex = cx - xh[h], ey = cy - yh[h];
                        double d = sqrt(ex * ex + ey * ey);
                        if (fabs(d - R) < H->tol) votes += 1;
                    }
                }
                if (accum) accum[lin] = votes;
                if (best_lin < 0 || votes > best_votes) {
                    best_lin = lin; best_votes = votes; bR = iR; bcy = icy; bcx = icx;
                }
            }
        }
    }
    peak[0] = bR; peak[1] = bcy; peak[2] = bcx; peak[3] = (int32_t)best_votes;
    /* circle -> transverse seed at R0 (Fig. 4) */
    {
        double R = H->R_lo + ((double)bR + 0.5) * H->bin_R;
        double cy = -H->half_xy + ((double)bcy + 0.5) * H->bin_xy;
        double cx = -H->half_xy + ((double)bcx + 0.5) * H->bin_xy;
        double cn = sqrt(cx * cx + cy * cy);
        double gamma = atan2(cy, cx);
        double cb = (g->R0 * g->R0 + cn * cn - R * R) / (2.0 * g->R0 * cn);
        if (cb > 1.0) cb = 1.0;
        if (cb < -1.0) cb = -1.0;
        double beta = acos(cb);
        /* q*Bz < 0: counter-clockwise seen from +z, outward crossing at gamma - beta */
        double sgn = ((double)charge * bz < 0.0) ? 1.0 : -1.0;
        double th = gamma - sgn * beta;
        double ex = g->R0 * cos(th), ey = g->R0 * sin(th);
        double pt = ORC_KAPPA * fabs(bz) * R;
        double px = sgn * pt * (-(ey - cy)) / R;
        double py = sgn * pt * (ex - cx) / R;
        ranges[0] = th - H->half_theta; ranges[1] = th + H->half_theta;
        ranges[2] = px - H->half_pt;    ranges[3] = px + H->half_pt;
        ranges[4] = py - H->half_pt;    ranges[5] = py + H->half_pt;
    }
    free(xh); free(yh);
}

/* ---- A1: dense per-wire drift table (sentinel -1 = no hit) ---------------- */
void orc_bin_event(const orc_geom *g, const orc_hits *hits, float *drift_of_wire)
{
    int i;
    for (i = 0; i < g->n_wires_total; ++i) drift_of_wire[i] = -1.0f;
    for (i = 0; i < hits->n_hits; ++i) drift_of_wire[hits->wire_id[i]] = hits->drift[i];
}
