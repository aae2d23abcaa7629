/*
 * p3t_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision CPU oracle for the soft-force half of the
 * P3T scheme of arXiv 1506.04553 (Iwasawa, Portegies Zwart, Makino).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code with the CUDA
 * path under paper_1506_04553_b200/csrc and neither includes the other.
 *
 * Citations are PAPER.md line numbers (L..) plus the equation they fall in.
 *
 *   O1  cutoff functions K (Eq. 12) and W (Eq. 16-17)
 *   O2  direct O(N^2) soft (and complementary hard) acceleration and
 *       potential (Eq. 5-8)
 *   O3  exact neighbour sets, brute force and sort-and-sweep (L138-140)
 *   O4  pointer-based Barnes-Hut octree, monopole + quadrupole (L138),
 *       opening parameter theta (L171), rule R-MAC / R-QUAD of DESIGN.md
 *   O6  hard acceleration (Eq. 7), its time derivative and the hard
 *       potential (Eq. 5) -- the NEXT row of SURVEY.md 8(f), pinned by
 *       tests/test_oracle_hard.py
 *   O7  one soft step under H_hard: drift of the isolated particles, fourth-order
 *       Hermite with block timesteps over the neighbour lists (L147, Eq. 18-20
 *       L152-163) -- rank 2 of SURVEY.md 8(f), pinned by tests/test_oracle_hermite.py
 *   O8  per-pair-class cutoffs (section 3.2.2.1): O2, O3, O6 and O4 with a class
 *       per body and (eps, r_in, r_cut, h) per kind of pair, unsplit BH-BH pairs --
 *       rank 3 of SURVEY.md 8(f), pinned by tests/test_oracle_classes.py
 *
 * Readings of the paper used here (each listed in DESIGN.md section 3):
 *   A1  Eq. 17's denominator is (gamma-1)^7 (as extracted it is (1-gamma)^7,
 *       which breaks Eq. 9; pinned by tests/test_oracle_cutoff.py).
 *   A3  acceleration is weighted by K, potential by W.
 *   A4  neighbour test is on the softened separation: s_ij < h.
 *   A13 the self term is excluded by index, not by distance.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md section 4.
 * Parity unpinned: the absolute tree-error level at a given theta (the paper
 * prints only whole-integration energy errors, Fig. 2-3); O4 is pinned by
 * theta=0 == O2, neighbour sets == O3, the (l/d)^3 error slope of the
 * acceleration AND of the potential, a = -grad phi of the accepted cells and
 * moment identities instead.  Also unpinned by nature: the exact form of the
 * step criterion Eq. 18 (reading A22; pins S1-S10 hold for any criterion of
 * the right dimension).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ O1 -- */

/* Eq. 12 (L85): K(x) = 0 (x<0); -20x^7+70x^6-84x^5+35x^4 (0<=x<1); 1 (1<=x) */
double p3t_oracle_K(double x)
{
    if (x < 0.0) return 0.0;
    if (x >= 1.0) return 1.0;
    double x2 = x * x, x4 = x2 * x2;
    return -20.0 * x4 * x2 * x + 70.0 * x4 * x2 - 84.0 * x4 * x + 35.0 * x4;
}

/* Eq. 16 first branch (L102): slope of W below gamma. */
double p3t_oracle_Cin(double g)
{
    double g2 = g * g, g3 = g2 * g, g4 = g2 * g2, g5 = g4 * g, g6 = g3 * g3;
    double glog = (g > 0.0) ? 60.0 * g3 * log(g) : 0.0; /* g^3 ln g -> 0 */
    double num = 7.0 * (g6 - 9.0 * g5 + 45.0 * g4 - glog - 45.0 * g2 + 9.0 * g - 1.0);
    double gm1 = g - 1.0, gm1_2 = gm1 * gm1, gm1_4 = gm1_2 * gm1_2;
    return num / (3.0 * gm1_4 * gm1_2 * gm1);
}

/* Eq. 17 (L104), denominator read as (gamma-1)^7 (reading A1). */
double p3t_oracle_G(double y, double g)
{
    double g2 = g * g, g3 = g2 * g, g4 = g2 * g2, g5 = g4 * g, g6 = g3 * g3, g7 = g6 * g;
    double y2 = y * y, y3 = y2 * y, y4 = y2 * y2, y5 = y4 * y, y6 = y3 * y3, y7 = y6 * y;
    double ylogy = (y > 0.0) ? y * log(y) : 0.0;
    double num = -(10.0 / 3.0) * y7
               + 14.0 * (g + 1.0) * y6
               - 21.0 * (g2 + 3.0 * g + 1.0) * y5
               + (35.0 * (g3 + 9.0 * g2 + 9.0 * g + 1.0) / 3.0) * y4
               - 70.0 * (g3 + 3.0 * g2 + g) * y3
               + 210.0 * (g3 + g2) * y2
               - 140.0 * g3 * ylogy
               + (g7 - 7.0 * g6 + 21.0 * g5 - 35.0 * g4);
    double gm1 = g - 1.0, gm1_2 = gm1 * gm1, gm1_4 = gm1_2 * gm1_2;
    return num / (gm1_4 * gm1_2 * gm1);
}

/* Eq. 16 (L102): W(y; gamma), three branches exactly as printed. */
double p3t_oracle_W(double y, double g)
{
    if (y < g) return p3t_oracle_Cin(g) * y;
    if (y < 1.0) return p3t_oracle_G(y, g) + (1.0 - p3t_oracle_G(1.0, g)) * y;
    return 1.0;
}

/* Eq. 13-15 (L87-94): x = (y-gamma)/(1-gamma), y = s/r_cut, gamma = r_in/r_cut. */
static inline void pair_weights(double s, double r_in, double r_out, double *K, double *W)
{
    double y = s / r_out;
    double g = r_in / r_out;
    double x = (y - g) / (1.0 - g);
    *K = p3t_oracle_K(x);
    *W = p3t_oracle_W(y, g);
}

/* exported for the tests: K and W as functions of the softened separation */
void p3t_oracle_pair_weights(double s, double r_in, double r_out, double *K, double *W)
{
    pair_weights(s, r_in, r_out, K, W);
}

/* ------------------------------------------------------------------ O2 -- */

/* Neumaier compensated accumulator. */
typedef struct { double s, c; } nsum;
static inline void nadd(nsum *a, double v)
{
    double t = a->s + v;
    if (fabs(a->s) >= fabs(v)) a->c += (a->s - t) + v;
    else                       a->c += (v - t) + a->s;
    a->s = t;
}
static inline double nval(const nsum *a) { return a->s + a->c; }

/*
 * Direct sum, Eq. 6 and 8 (L55, L65), per unit mass of particle i (L108-109):
 *   a_soft,i  = - sum_{j!=i} m_j K(s_ij) (q_i - q_j) / s_ij^3
 *   phi_soft,i= - sum_{j!=i} m_j W(s_ij) / s_ij
 * and the complementary hard terms of Eq. 5 and 7 (L53, L63) with (1-K),
 * (1-W).  s_ij = sqrt(|q_ij|^2 + eps^2) (Eq. 2).  j != i by index.
 * subset == NULL means i = 0..ns-1.  Output arrays may be NULL.
 */
void p3t_oracle_direct(int64_t n, const double *m, const double *q,
                       double eps, double r_in, double r_out,
                       int64_t ns, const int64_t *subset,
                       double *acc_soft, double *pot_soft,
                       double *acc_hard, double *pot_hard)
{
    const double eps2 = eps * eps;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ns; ++k) {
        int64_t i = subset ? subset[k] : k;
        double xi = q[3 * i], yi = q[3 * i + 1], zi = q[3 * i + 2];
        nsum as[3] = {{0, 0}, {0, 0}, {0, 0}}, ah[3] = {{0, 0}, {0, 0}, {0, 0}};
        nsum ps = {0, 0}, ph = {0, 0};
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = xi - q[3 * j], dy = yi - q[3 * j + 1], dz = zi - q[3 * j + 2];
            double s2 = dx * dx + dy * dy + dz * dz + eps2;
            double s = sqrt(s2);
            double K, W;
            if (s >= r_out) { K = 1.0; W = 1.0; }     /* Eq. 12/16 third branches */
            else pair_weights(s, r_in, r_out, &K, &W);
            double mr1 = m[j] / s;
            double mr3 = mr1 / s2;
            nadd(&as[0], -mr3 * K * dx); nadd(&as[1], -mr3 * K * dy); nadd(&as[2], -mr3 * K * dz);
            nadd(&ps, -mr1 * W);
            nadd(&ah[0], -mr3 * (1.0 - K) * dx); nadd(&ah[1], -mr3 * (1.0 - K) * dy);
            nadd(&ah[2], -mr3 * (1.0 - K) * dz);
            nadd(&ph, -mr1 * (1.0 - W));
        }
        if (acc_soft) for (int d = 0; d < 3; ++d) acc_soft[3 * k + d] = nval(&as[d]);
        if (pot_soft) pot_soft[k] = nval(&ps);
        if (acc_hard) for (int d = 0; d < 3; ++d) acc_hard[3 * k + d] = nval(&ah[d]);
        if (pot_hard) pot_hard[k] = nval(&ph);
    }
}

/* ------------------------------------------------------------------ O6 -- */

/* dK/dx of Eq. 12 (L85) on 0 <= x < 1, 0 elsewhere: the derivative of the printed polynomial,
 * -140x^6 + 420x^5 - 420x^4 + 140x^3 = 140 x^3 (1-x)^3 (factored: no cancellation near x = 1). */
double p3t_oracle_dKdx(double x)
{
    if (x < 0.0 || x >= 1.0) return 0.0;
    double u = x * (1.0 - x);
    return 140.0 * u * u * u;
}

/*
 * Hard acceleration and its time derivative (jerk), the quantities the Hermite part integrates (Eq. 7;
 * procedure step 3 L147), per unit mass of i, over ALL j != i:
 *   a_i = - sum_j m_j (1 - K(s)) q_ij / s^3
 *   j_i = d a_i / dt with q_ij -> q_ij + v_ij t:  ds/dt = (q_ij . v_ij) / s,
 *       = - sum_j m_j [ (1 - K) ( v_ij / s^3 - 3 (q.v) q_ij / s^5 ) - (dK/ds) ((q.v)/s) q_ij / s^3 ],
 *   dK/ds = dK/dx / (r_out (1 - gamma))   (x of Eq. 13).
 * (The paper gives Eq. 7 only; the jerk is its time derivative written out.)
 */
void p3t_oracle_hard(int64_t n, const double *m, const double *q, const double *v,
                     double eps, double r_in, double r_out,
                     int64_t ns, const int64_t *subset, double *acc, double *jerk, double *pot)
{
    const double eps2 = eps * eps, g = r_in / r_out;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ns; ++k) {
        int64_t i = subset ? subset[k] : k;
        nsum a[3] = {{0, 0}, {0, 0}, {0, 0}}, jk[3] = {{0, 0}, {0, 0}, {0, 0}}, ph = {0, 0};
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[3], w[3];
            for (int c = 0; c < 3; ++c) { d[c] = q[3 * i + c] - q[3 * j + c]; w[c] = v[3 * i + c] - v[3 * j + c]; }
            double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + eps2;
            double s = sqrt(s2);
            if (s >= r_out) continue;                       /* 1 - K = 1 - W = 0 (Eq. 12/16 third branches) */
            double K, W;
            pair_weights(s, r_in, r_out, &K, &W);
            double x = (s / r_out - g) / (1.0 - g);
            double dKds = p3t_oracle_dKdx(x) / (r_out * (1.0 - g));
            double qv = d[0] * w[0] + d[1] * w[1] + d[2] * w[2];
            double mr3 = m[j] / (s2 * s);
            for (int c = 0; c < 3; ++c) {
                nadd(&a[c], -mr3 * (1.0 - K) * d[c]);
                nadd(&jk[c], -mr3 * ((1.0 - K) * (w[c] - 3.0 * qv * d[c] / s2) - dKds * (qv / s) * d[c]));
            }
            nadd(&ph, -(m[j] / s) * (1.0 - W));
        }
        for (int c = 0; c < 3; ++c) {
            if (acc) acc[3 * k + c] = nval(&a[c]);
            if (jerk) jerk[3 * k + c] = nval(&jk[c]);
        }
        if (pot) pot[k] = nval(&ph);
    }
}

/* ------------------------------------------------------------------ O7 -- */

/*
 * Integration of all particles over one soft step T under H_hard (procedure step 3, L147; GPU procedure steps 5-6,
 * section 2.2): particles with an empty neighbour list drift, x += T v; the others are integrated with the
 * fourth-order Hermite scheme with block timesteps, the force being Eq. 7 (L63) summed over the particle's neighbour
 * list (offset/list, fixed during the step; 1 - K = 0 beyond r_out <= h so the list sum is the full hard force as long
 * as nobody outside the list comes within r_out).  Readings (A21-A24):
 *  - time is counted in ticks of T / 2^40; a particle's step is a power of two of ticks, at most T / 2^log2_div
 *    (Delta t_max, L150), the largest one not above the criterion that divides the particle's current time
 *    (block steps); never below one tick (returned in floor_hits);
 *  - first step: Eq. 20 (L163), dt = eta_s sqrt((|a|^2 + a0^2) / |a1|^2); later steps: Eq. 18 (L152) read as
 *    Aarseth's criterion with |a| replaced by sqrt(|a|^2 + a0^2),
 *        dt = eta sqrt( (sqrt(|a|^2 + a0^2) |a2| + |a1|^2) / (|a1| |a3| + |a2|^2) )
 *    (the printed denominator |a||a3| is not a time squared); a2, a3 from the Hermite interpolation, a2 taken at
 *    the end of the step (a2 + dt a3); a vanishing denominator gives Delta t_max;
 *  - predictor x_p = x + v dt + a dt^2/2 + a1 dt^3/6, v_p = v + a dt + a1 dt^2/2 for the active particle and for
 *    each of its neighbours from that neighbour's own last time; corrector
 *        a2 = (-6 (a - a_n) - dt (4 a1 + 2 a1_n)) / dt^2,  a3 = (12 (a - a_n) + 6 dt (a1 + a1_n)) / dt^3,
 *        x = x_p + a2 dt^4/24 + a3 dt^5/120,  v = v_p + a2 dt^3/6 + a3 dt^4/24   (Makino & Aarseth 1992);
 *  - all active particles of a block are evaluated from the state before the block, then corrected together.
 * Sums run in list order, plain fp64.  q, v are updated in place.  nstep[i] (may be NULL) receives the number of
 * Hermite steps of particle i.  Returns the number of blocks, or -1 when more than max_blocks would be needed (a0 = 0
 * lets Eq. 18 collapse at the edge of the cutoff sphere, L152; q, v are then left mid-step).
 */
#define O7_TICK_BITS 40

static void o7_force(int64_t i, const double *m, const double *xp, const double *vp,
                     const int64_t *offset, const int32_t *list,
                     double eps2, double r_in, double r_out, double *a, double *a1)
{
    const double g = r_in / r_out;
    for (int c = 0; c < 3; ++c) a[c] = a1[c] = 0.0;
    for (int64_t e = offset[i]; e < offset[i + 1]; ++e) {
        int64_t j = list[e];
        const double *xj = xp + 3 * (e - offset[i] + 1), *vj = vp + 3 * (e - offset[i] + 1);
        double d[3], w[3];
        for (int c = 0; c < 3; ++c) { d[c] = xp[c] - xj[c]; w[c] = vp[c] - vj[c]; }
        double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + eps2;
        double s = sqrt(s2);
        if (s >= r_out) continue;
        double K, W;
        pair_weights(s, r_in, r_out, &K, &W);
        double x = (s / r_out - g) / (1.0 - g);
        double dKds = p3t_oracle_dKdx(x) / (r_out * (1.0 - g));
        double qv = d[0] * w[0] + d[1] * w[1] + d[2] * w[2];
        double mr3 = m[j] / (s2 * s);
        for (int c = 0; c < 3; ++c) {
            a[c] += -mr3 * (1.0 - K) * d[c];
            a1[c] += -mr3 * ((1.0 - K) * (w[c] - 3.0 * qv * d[c] / s2) - dKds * (qv / s) * d[c]);
        }
    }
}

static double o7_norm(const double *u) { return sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]); }

/* largest power of two of ticks <= crit (a time), <= max_ticks, dividing t; at least one tick */
static int64_t o7_quantise(double crit, double tick, int64_t max_ticks, int64_t t, int64_t *floor_hits)
{
    int64_t dt;
    double ct = crit / tick;
    if (!(ct < (double)max_ticks)) dt = max_ticks;          /* also NaN, inf */
    else if (ct < 1.0) { dt = 1; if (floor_hits) ++*floor_hits; }
    else { int e; frexp(ct, &e); dt = (int64_t)1 << (e - 1); }
    while (t % dt) dt >>= 1;
    return dt;
}

int64_t p3t_oracle_hermite(int64_t n, const double *m, double *q, double *v,
                           double eps, double r_in, double r_out,
                           const int64_t *offset, const int32_t *list,
                           double T, int log2_div, double eta, double eta_s, double a0, int64_t max_blocks,
                           int64_t *nstep, int64_t *floor_hits)
{
    const double eps2 = eps * eps;
    const int64_t total = (int64_t)1 << O7_TICK_BITS, max_ticks = total >> log2_div;
    const double tick = T / (double)total;
    int64_t *t = calloc((size_t)n, sizeof *t), *dt = calloc((size_t)n, sizeof *dt);
    double *a = calloc((size_t)3 * n, sizeof *a), *a1 = calloc((size_t)3 * n, sizeof *a1);
    double *an = calloc((size_t)3 * n, sizeof *an), *a1n = calloc((size_t)3 * n, sizeof *a1n);
    int64_t maxl = 0, nblocks = 0;
    if (floor_hits) *floor_hits = 0;
    for (int64_t i = 0; i < n; ++i) if (offset[i + 1] - offset[i] > maxl) maxl = offset[i + 1] - offset[i];
    double *xp = malloc((size_t)3 * (maxl + 1) * sizeof *xp), *vp = malloc((size_t)3 * (maxl + 1) * sizeof *vp);

    /* t = 0: forces from the current state, first steps from Eq. 20 */
    for (int64_t i = 0; i < n; ++i) {
        if (nstep) nstep[i] = 0;
        if (offset[i + 1] == offset[i]) continue;
        for (int c = 0; c < 3; ++c) { xp[c] = q[3 * i + c]; vp[c] = v[3 * i + c]; }
        for (int64_t e = offset[i]; e < offset[i + 1]; ++e)
            for (int c = 0; c < 3; ++c) {
                xp[3 * (e - offset[i] + 1) + c] = q[3 * (int64_t)list[e] + c];
                vp[3 * (e - offset[i] + 1) + c] = v[3 * (int64_t)list[e] + c];
            }
        o7_force(i, m, xp, vp, offset, list, eps2, r_in, r_out, a + 3 * i, a1 + 3 * i);
        double na = o7_norm(a + 3 * i), n1 = o7_norm(a1 + 3 * i);
        double crit = n1 > 0.0 ? eta_s * sqrt((na * na + a0 * a0) / (n1 * n1)) : INFINITY;
        dt[i] = o7_quantise(crit, tick, max_ticks, 0, floor_hits);
    }
    for (;;) {
        int64_t tn = INT64_MAX;
        for (int64_t i = 0; i < n; ++i)
            if (offset[i + 1] > offset[i] && t[i] < total && t[i] + dt[i] < tn) tn = t[i] + dt[i];
        if (tn == INT64_MAX) break;
        if (++nblocks > max_blocks) { nblocks = -1; break; }
        /* evaluate every active particle from the state before the block */
        for (int64_t i = 0; i < n; ++i) {
            if (offset[i + 1] == offset[i] || t[i] + dt[i] != tn) continue;
            for (int64_t k = 0; k <= offset[i + 1] - offset[i]; ++k) {
                int64_t j = k ? (int64_t)list[offset[i] + k - 1] : i;
                double h = (double)(tn - t[j]) * tick;
                for (int c = 0; c < 3; ++c) {
                    double A = a[3 * j + c], J = a1[3 * j + c];
                    xp[3 * k + c] = q[3 * j + c] + h * (v[3 * j + c] + h * (A / 2.0 + h * (J / 6.0)));
                    vp[3 * k + c] = v[3 * j + c] + h * (A + h * (J / 2.0));
                }
            }
            o7_force(i, m, xp, vp, offset, list, eps2, r_in, r_out, an + 3 * i, a1n + 3 * i);
        }
        /* correct them together */
        for (int64_t i = 0; i < n; ++i) {
            if (offset[i + 1] == offset[i] || t[i] + dt[i] != tn) continue;
            double h = (double)dt[i] * tick, a2[3], a3[3], a2e[3];
            for (int c = 0; c < 3; ++c) {
                double A = a[3 * i + c], J = a1[3 * i + c], An = an[3 * i + c], Jn = a1n[3 * i + c];
                a2[c] = (-6.0 * (A - An) - h * (4.0 * J + 2.0 * Jn)) / (h * h);
                a3[c] = (12.0 * (A - An) + 6.0 * h * (J + Jn)) / (h * h * h);
                double x_p = q[3 * i + c] + h * (v[3 * i + c] + h * (A / 2.0 + h * (J / 6.0)));
                double v_p = v[3 * i + c] + h * (A + h * (J / 2.0));
                q[3 * i + c] = x_p + h * h * h * h * (a2[c] / 24.0 + h * a3[c] / 120.0);
                v[3 * i + c] = v_p + h * h * h * (a2[c] / 6.0 + h * a3[c] / 24.0);
                a2e[c] = a2[c] + h * a3[c];
                a[3 * i + c] = An; a1[3 * i + c] = Jn;
            }
            t[i] = tn;
            if (nstep) ++nstep[i];
            double na = o7_norm(a + 3 * i), n1 = o7_norm(a1 + 3 * i), n2 = o7_norm(a2e), n3 = o7_norm(a3);
            double den = n1 * n3 + n2 * n2;
            double crit = den > 0.0 ? eta * sqrt((sqrt(na * na + a0 * a0) * n2 + n1 * n1) / den) : INFINITY;
            dt[i] = o7_quantise(crit, tick, max_ticks, tn, floor_hits);
        }
    }
    for (int64_t i = 0; i < n && nblocks >= 0; ++i)
        if (offset[i + 1] == offset[i])
            for (int c = 0; c < 3; ++c) q[3 * i + c] += T * v[3 * i + c];
    free(t); free(dt); free(a); free(a1); free(an); free(a1n); free(xp); free(vp);
    return nblocks;
}

/* ------------------------------------------------------------------ O3 -- */

/*
 * Exact neighbour sets L_i = { j != i : s_ij < h } (L138-140; reading A4),
 * brute force.  plain != 0 switches to the plain-distance variant
 * |q_ij| < h.  Two passes by the caller: list == NULL -> only count[k].
 * With list != NULL, offset[ns+1] (exclusive prefix of count) says where
 * each list goes; entries are ascending in j.  Pairs with |s/h - 1| < band
 * are additionally recorded in band_pairs (k, j) up to band_cap; the number
 * of such pairs is returned.
 */
int64_t p3t_oracle_neighbours(int64_t n, const double *q, double eps, double h, int plain,
                              int64_t ns, const int64_t *subset,
                              int64_t *count, const int64_t *offset, int32_t *list,
                              double band, int64_t *band_pairs, int64_t band_cap)
{
    const double eps2 = plain ? 0.0 : eps * eps;
    int64_t nband = 0;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ns; ++k) {
        int64_t i = subset ? subset[k] : k;
        double xi = q[3 * i], yi = q[3 * i + 1], zi = q[3 * i + 2];
        int64_t c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = xi - q[3 * j], dy = yi - q[3 * j + 1], dz = zi - q[3 * j + 2];
            double s = sqrt(dx * dx + dy * dy + dz * dz + eps2);
            if (s < h) {
                if (list) list[offset[k] + c] = (int32_t)j;
                ++c;
            }
            if (band > 0.0 && fabs(s / h - 1.0) < band) {
                int64_t slot;
#pragma omp atomic capture
                slot = nband++;
                if (band_pairs && slot < band_cap) { band_pairs[2 * slot] = k; band_pairs[2 * slot + 1] = j; }
            }
        }
        if (count) count[k] = c;
    }
    return nband;
}

/*
 * Same sets for all i by sort-and-sweep along x (for N too large for the
 * O(N^2) loop).  Cross-checked against p3t_oracle_neighbours in the tests.
 * order[] must hold the particle indices sorted by ascending x (the caller
 * sorts).  Same two-pass convention as above; entries ascending in j.
 */
static int cmp_i32(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}
void p3t_oracle_neighbours_sweep(int64_t n, const double *q, double eps, double h, int plain,
                                 const int64_t *order,
                                 int64_t *count, const int64_t *offset, int32_t *list)
{
    const double eps2 = plain ? 0.0 : eps * eps;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t r = 0; r < n; ++r) {
        int64_t i = order[r];
        double xi = q[3 * i], yi = q[3 * i + 1], zi = q[3 * i + 2];
        int64_t c = 0;
        for (int dir = -1; dir <= 1; dir += 2) {
            for (int64_t t = r + dir; t >= 0 && t < n; t += dir) {
                int64_t j = order[t];
                double dx = xi - q[3 * j];
                if (fabs(dx) >= h) break; /* |q_ij| >= |dx| >= h  =>  s >= h */
                double dy = yi - q[3 * j + 1], dz = zi - q[3 * j + 2];
                double s = sqrt(dx * dx + dy * dy + dz * dz + eps2);
                if (s < h) {
                    if (list) list[offset[i] + c] = (int32_t)j;
                    ++c;
                }
            }
        }
        if (count) count[i] = c;
        if (list && c > 1) qsort(list + offset[i], (size_t)c, sizeof(int32_t), cmp_i32);
    }
}

/* ------------------------------------------------------------------ O4 -- */

/*
 * Pointer-based Barnes-Hut octree (deliberately not Morton/sort based).
 *  1. root cube: centre = midpoint of the position AABB, side = largest
 *     extent * (1 + 1e-6)
 *  2. a cell with more than nleaf bodies splits into octants about its
 *     geometric centre until <= nleaf or depth == max_depth
 *  3. post-order moments: M, centre of mass c, traceful quadrupole
 *     Q_ab = sum m (x-c)_a (x-c)_b, tight AABB of the bodies
 *  4. walk per target i with box B_i (degenerate = the particle, or a box
 *     supplied by the caller): accept cell C iff   (rule R-MAC)
 *        theta > 0  and  d(B, c_C) > l_C/theta + |c_C - g_C|
 *                   and  D(B, AABB_C) >= h
 *     else leaf -> direct terms (O2 formulas, j != i), internal -> recurse
 *  5. accepted cell (rule R-QUAD, K = W = 1, Plummer-softened):
 *        R = q_i - c, s^2 = |R|^2 + eps^2
 *        phi += -M/s - 1/2 [ 3 R'QR / s^5 - tr Q / s^3 ]
 *        a   += -M R/s^3 + 3 QR/s^5 - 15/2 (R'QR) R/s^7 + 3/2 trQ R/s^5
 *     (second-order Taylor expansion of -sum m/sqrt(|R-x|^2+eps^2) about c)
 *  6. neighbour candidates: every body met in an opened leaf with s < h
 */
typedef struct {
    double g[3], side;      /* cube geometric centre and side */
    double M, c[3], Q[6];   /* xx yy zz xy xz yz */
    double bmin[3], bmax[3];
    int32_t child[8];
    int32_t first, count;   /* range in tree->perm (all bodies of the subtree) */
    int32_t leaf, level;
} onode;

typedef struct {
    onode *node; int64_t nnode, cap;
    int32_t *perm;          /* body indices, subtree-contiguous */
    int64_t n;
    const double *m, *q;
    int nleaf, max_depth;
} otree;

static int32_t new_node(otree *t)
{
    if (t->nnode == t->cap) {
        t->cap = t->cap ? 2 * t->cap : 1024;
        t->node = (onode *)realloc(t->node, (size_t)t->cap * sizeof(onode));
    }
    memset(&t->node[t->nnode], 0, sizeof(onode));
    for (int k = 0; k < 8; ++k) t->node[t->nnode].child[k] = -1;
    return (int32_t)t->nnode++;
}

static int32_t build_rec(otree *t, int32_t first, int32_t count, const double g[3], double side, int level,
                         int32_t *scratch)
{
    int32_t id = new_node(t);
    {
        onode *nd = &t->node[id];
        nd->g[0] = g[0]; nd->g[1] = g[1]; nd->g[2] = g[2]; nd->side = side;
        nd->first = first; nd->count = count; nd->level = level;
        nd->leaf = (count <= t->nleaf || level >= t->max_depth);
    }
    if (!t->node[id].leaf) {
        /* partition perm[first, first+count) into octants: bit0 = x, bit1 = y, bit2 = z */
        int32_t cnt[8] = {0}, start[8];
        for (int32_t k = 0; k < count; ++k) {
            int32_t b = t->perm[first + k];
            int o = (t->q[3 * b] >= g[0]) | ((t->q[3 * b + 1] >= g[1]) << 1) | ((t->q[3 * b + 2] >= g[2]) << 2);
            cnt[o]++;
        }
        start[0] = 0;
        for (int o = 1; o < 8; ++o) start[o] = start[o - 1] + cnt[o - 1];
        int32_t pos[8];
        memcpy(pos, start, sizeof pos);
        for (int32_t k = 0; k < count; ++k) {
            int32_t b = t->perm[first + k];
            int o = (t->q[3 * b] >= g[0]) | ((t->q[3 * b + 1] >= g[1]) << 1) | ((t->q[3 * b + 2] >= g[2]) << 2);
            scratch[first + pos[o]++] = b;
        }
        memcpy(t->perm + first, scratch + first, (size_t)count * sizeof(int32_t));
        for (int o = 0; o < 8; ++o) {
            if (!cnt[o]) continue;
            double cg[3] = { g[0] + ((o & 1) ? 0.25 : -0.25) * side,
                             g[1] + ((o & 2) ? 0.25 : -0.25) * side,
                             g[2] + ((o & 4) ? 0.25 : -0.25) * side };
            int32_t ch = build_rec(t, first + start[o], cnt[o], cg, 0.5 * side, level + 1, scratch);
            t->node[id].child[o] = ch; /* re-index: node array may have moved */
        }
    }
    /* post-order moments (step 3) */
    onode *nd = &t->node[id];
    double M = 0, c[3] = {0, 0, 0};
    for (int d = 0; d < 3; ++d) { nd->bmin[d] = INFINITY; nd->bmax[d] = -INFINITY; }
    if (nd->leaf) {
        for (int32_t k = 0; k < count; ++k) {
            int32_t b = t->perm[first + k];
            M += t->m[b];
            for (int d = 0; d < 3; ++d) {
                c[d] += t->m[b] * t->q[3 * b + d];
                nd->bmin[d] = fmin(nd->bmin[d], t->q[3 * b + d]);
                nd->bmax[d] = fmax(nd->bmax[d], t->q[3 * b + d]);
            }
        }
        for (int d = 0; d < 3; ++d) c[d] = (M > 0) ? c[d] / M : g[d];
        double Q[6] = {0};
        for (int32_t k = 0; k < count; ++k) {
            int32_t b = t->perm[first + k];
            double r[3] = { t->q[3 * b] - c[0], t->q[3 * b + 1] - c[1], t->q[3 * b + 2] - c[2] };
            double mb = t->m[b];
            Q[0] += mb * r[0] * r[0]; Q[1] += mb * r[1] * r[1]; Q[2] += mb * r[2] * r[2];
            Q[3] += mb * r[0] * r[1]; Q[4] += mb * r[0] * r[2]; Q[5] += mb * r[1] * r[2];
        }
        memcpy(nd->Q, Q, sizeof Q);
    } else {
        for (int o = 0; o < 8; ++o) {
            if (nd->child[o] < 0) continue;
            const onode *ch = &t->node[nd->child[o]];
            M += ch->M;
            for (int d = 0; d < 3; ++d) {
                c[d] += ch->M * ch->c[d];
                nd->bmin[d] = fmin(nd->bmin[d], ch->bmin[d]);
                nd->bmax[d] = fmax(nd->bmax[d], ch->bmax[d]);
            }
        }
        for (int d = 0; d < 3; ++d) c[d] = (M > 0) ? c[d] / M : g[d];
        double Q[6] = {0};
        for (int o = 0; o < 8; ++o) { /* parallel-axis shift of each child's Q to the parent's c */
            if (nd->child[o] < 0) continue;
            const onode *ch = &t->node[nd->child[o]];
            double r[3] = { ch->c[0] - c[0], ch->c[1] - c[1], ch->c[2] - c[2] };
            Q[0] += ch->Q[0] + ch->M * r[0] * r[0]; Q[1] += ch->Q[1] + ch->M * r[1] * r[1];
            Q[2] += ch->Q[2] + ch->M * r[2] * r[2]; Q[3] += ch->Q[3] + ch->M * r[0] * r[1];
            Q[4] += ch->Q[4] + ch->M * r[0] * r[2]; Q[5] += ch->Q[5] + ch->M * r[1] * r[2];
        }
        memcpy(nd->Q, Q, sizeof Q);
    }
    nd->M = M; nd->c[0] = c[0]; nd->c[1] = c[1]; nd->c[2] = c[2];
    return id;
}

void *p3t_oracle_tree_build(int64_t n, const double *m, const double *q, int nleaf, int max_depth)
{
    otree *t = (otree *)calloc(1, sizeof(otree));
    t->n = n; t->m = m; t->q = q; t->nleaf = nleaf; t->max_depth = max_depth;
    t->perm = (int32_t *)malloc((size_t)n * sizeof(int32_t));
    int32_t *scratch = (int32_t *)malloc((size_t)n * sizeof(int32_t));
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int64_t i = 0; i < n; ++i) {
        t->perm[i] = (int32_t)i;
        for (int d = 0; d < 3; ++d) { lo[d] = fmin(lo[d], q[3 * i + d]); hi[d] = fmax(hi[d], q[3 * i + d]); }
    }
    double g[3], side = 0;
    for (int d = 0; d < 3; ++d) { g[d] = 0.5 * (lo[d] + hi[d]); side = fmax(side, hi[d] - lo[d]); }
    side *= (1.0 + 1e-6);
    if (!(side > 0)) side = 1.0;
    build_rec(t, 0, (int32_t)n, g, side, 0, scratch);
    free(scratch);
    return t;
}

void p3t_oracle_tree_free(void *tree)
{
    otree *t = (otree *)tree;
    if (!t) return;
    free(t->node); free(t->perm); free(t);
}

int64_t p3t_oracle_tree_nnodes(const void *tree) { return ((const otree *)tree)->nnode; }

/* node k -> 32 doubles: g[3] side M c[3] Q[6] bmin[3] bmax[3] first count leaf level child[8] */
void p3t_oracle_tree_node(const void *tree, int64_t k, double *out)
{
    const onode *nd = &((const otree *)tree)->node[k];
    int p = 0;
    for (int d = 0; d < 3; ++d) out[p++] = nd->g[d];
    out[p++] = nd->side; out[p++] = nd->M;
    for (int d = 0; d < 3; ++d) out[p++] = nd->c[d];
    for (int d = 0; d < 6; ++d) out[p++] = nd->Q[d];
    for (int d = 0; d < 3; ++d) out[p++] = nd->bmin[d];
    for (int d = 0; d < 3; ++d) out[p++] = nd->bmax[d];
    out[p++] = nd->first; out[p++] = nd->count; out[p++] = nd->leaf; out[p++] = nd->level;
    for (int d = 0; d < 8; ++d) out[p++] = nd->child[d];
}
void p3t_oracle_tree_perm(const void *tree, int32_t *perm)
{
    const otree *t = (const otree *)tree;
    memcpy(perm, t->perm, (size_t)t->n * sizeof(int32_t));
}

typedef struct {
    const otree *t;
    int64_t i;                 /* target index (self exclusion) */
    double x[3];               /* target position */
    double bmin[3], bmax[3];   /* target box B */
    double eps2, theta, h, r_in, r_out;
    int use_quad;
    nsum a[3], phi;
    int64_t n_pp, n_pc;
    int32_t *nbr; int64_t nbr_cap, nbr_n;
} walk_state;

static inline double box_point_dist2(const double lo[3], const double hi[3], const double p[3])
{
    double d2 = 0;
    for (int d = 0; d < 3; ++d) {
        double e = fmax(0.0, fmax(lo[d] - p[d], p[d] - hi[d]));
        d2 += e * e;
    }
    return d2;
}
static inline double box_box_dist2(const double lo[3], const double hi[3], const double lo2[3], const double hi2[3])
{
    double d2 = 0;
    for (int d = 0; d < 3; ++d) {
        double e = fmax(0.0, fmax(lo[d] - hi2[d], lo2[d] - hi[d]));
        d2 += e * e;
    }
    return d2;
}

static void walk_rec(walk_state *w, int32_t id)
{
    const onode *nd = &w->t->node[id];
    if (nd->count == 0) return;
    /* rule R-MAC */
    int accept = 0;
    if (w->theta > 0.0) {
        double delta = sqrt((nd->c[0] - nd->g[0]) * (nd->c[0] - nd->g[0]) +
                            (nd->c[1] - nd->g[1]) * (nd->c[1] - nd->g[1]) +
                            (nd->c[2] - nd->g[2]) * (nd->c[2] - nd->g[2]));
        double rc = nd->side / w->theta + delta;
        double d2 = box_point_dist2(w->bmin, w->bmax, nd->c);
        double D2 = box_box_dist2(w->bmin, w->bmax, nd->bmin, nd->bmax);
        accept = (d2 > rc * rc) && (D2 >= w->h * w->h);
    }
    if (accept) {
        /* rule R-QUAD */
        double R[3] = { w->x[0] - nd->c[0], w->x[1] - nd->c[1], w->x[2] - nd->c[2] };
        double s2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2] + w->eps2;
        double s = sqrt(s2), s3 = s * s2, s5 = s3 * s2, s7 = s5 * s2;
        const double *Q = nd->Q;
        double phi = -nd->M / s;
        double a[3] = { -nd->M * R[0] / s3, -nd->M * R[1] / s3, -nd->M * R[2] / s3 };
        if (w->use_quad) {
            double QR[3] = { Q[0] * R[0] + Q[3] * R[1] + Q[4] * R[2],
                             Q[3] * R[0] + Q[1] * R[1] + Q[5] * R[2],
                             Q[4] * R[0] + Q[5] * R[1] + Q[2] * R[2] };
            double RQR = R[0] * QR[0] + R[1] * QR[1] + R[2] * QR[2];
            double trQ = Q[0] + Q[1] + Q[2];
            phi += -0.5 * (3.0 * RQR / s5 - trQ / s3);
            for (int d = 0; d < 3; ++d)
                a[d] += 3.0 * QR[d] / s5 - 7.5 * RQR * R[d] / s7 + 1.5 * trQ * R[d] / s5;
        }
        for (int d = 0; d < 3; ++d) nadd(&w->a[d], a[d]);
        nadd(&w->phi, phi);
        w->n_pc++;
        return;
    }
    if (nd->leaf) {
        for (int32_t k = 0; k < nd->count; ++k) {
            int64_t j = w->t->perm[nd->first + k];
            if (j == w->i) continue;
            double dx = w->x[0] - w->t->q[3 * j], dy = w->x[1] - w->t->q[3 * j + 1], dz = w->x[2] - w->t->q[3 * j + 2];
            double s2 = dx * dx + dy * dy + dz * dz + w->eps2;
            double s = sqrt(s2);
            double K, W;
            if (s >= w->r_out) { K = 1.0; W = 1.0; }
            else pair_weights(s, w->r_in, w->r_out, &K, &W);
            double mr1 = w->t->m[j] / s, mr3 = mr1 / s2;
            nadd(&w->a[0], -mr3 * K * dx); nadd(&w->a[1], -mr3 * K * dy); nadd(&w->a[2], -mr3 * K * dz);
            nadd(&w->phi, -mr1 * W);
            w->n_pp++;
            if (s < w->h) {
                if (w->nbr && w->nbr_n < w->nbr_cap) w->nbr[w->nbr_n] = (int32_t)j;
                w->nbr_n++;
            }
        }
        return;
    }
    for (int o = 0; o < 8; ++o)
        if (nd->child[o] >= 0) walk_rec(w, nd->child[o]);
}

/*
 * Walk for targets subset[0..ns) (NULL -> 0..ns-1).  box == NULL: each target's
 * box is the particle itself; else box[6k..6k+5] = (min xyz, max xyz) of the
 * group the target belongs to.  nbr: per-target slabs of nbr_stride entries
 * (NULL to skip); nbr_count[k] is the true count even if it exceeds the slab.
 * counts[2k], counts[2k+1] = p-p and p-c interactions of target k.
 */
void p3t_oracle_tree_walk(const void *tree, double eps, double theta, double r_in, double r_out, double h,
                          int use_quad, int64_t ns, const int64_t *subset, const double *box,
                          double *acc, double *pot, int64_t *counts,
                          int32_t *nbr, int64_t nbr_stride, int64_t *nbr_count)
{
    const otree *t = (const otree *)tree;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t k = 0; k < ns; ++k) {
        walk_state w;
        memset(&w, 0, sizeof w);
        w.t = t; w.i = subset ? subset[k] : k;
        for (int d = 0; d < 3; ++d) {
            w.x[d] = t->q[3 * w.i + d];
            w.bmin[d] = box ? box[6 * k + d] : w.x[d];
            w.bmax[d] = box ? box[6 * k + 3 + d] : w.x[d];
        }
        w.eps2 = eps * eps; w.theta = theta; w.h = h; w.r_in = r_in; w.r_out = r_out; w.use_quad = use_quad;
        w.nbr = nbr ? nbr + k * nbr_stride : NULL; w.nbr_cap = nbr_stride;
        walk_rec(&w, 0);
        if (acc) for (int d = 0; d < 3; ++d) acc[3 * k + d] = nval(&w.a[d]);
        if (pot) pot[k] = nval(&w.phi);
        if (counts) { counts[2 * k] = w.n_pp; counts[2 * k + 1] = w.n_pc; }
        if (nbr_count) nbr_count[k] = w.nbr_n;
        if (w.nbr && w.nbr_n > 1)
            qsort(w.nbr, (size_t)(w.nbr_n < w.nbr_cap ? w.nbr_n : w.nbr_cap), sizeof(int32_t), cmp_i32);
    }
}

/* ------------------------------------------------------------------ O8 -- */

/*
 * Per-pair-class cutoffs (section 3.2.2.1: "three values for the cut off radius with respect to three different
 * kinds of interactions"): every body carries a class, 0 = field star (FS) or 1 = black hole (BH); the kind of a pair is
 * k = cls_i + cls_j (0: FS-FS, 1: BH-FS, 2: BH-BH) and each kind has its own softening, cutoff radii and neighbour
 * radius, tab[4 k .. 4 k + 3] = (eps, r_in, r_cut, h).  A kind whose r_cut is +infinity is NOT SPLIT (L287: "the force
 * is not split and F_soft = 0 ... integrated with the pure Hermite scheme"): K = W = 0 in the soft sums, 1 - K = 1 - W
 * = 1 in the hard sums at every separation, and the two bodies are always in each other's neighbour list.  Everything
 * else is O2 / O3 / O6 / O4 with the pair's own numbers.  With all classes 0 these functions reduce to the ones above.
 */
typedef struct { double eps2, r_in, r_out, h; int unsplit; } pairprm;

static inline pairprm pair_of(const double *tab, const uint8_t *cls, int64_t i, int64_t j)
{
    const double *t = tab + 4 * ((int)cls[i] + (int)cls[j]);
    pairprm p = { t[0] * t[0], t[1], t[2], t[3], isinf(t[2]) ? 1 : 0 };
    return p;
}

/* K, W of a pair at softened separation s */
static inline void pair_weights_cls(const pairprm *p, double s, double *K, double *W)
{
    if (p->unsplit) { *K = 0.0; *W = 0.0; }
    else if (s >= p->r_out) { *K = 1.0; *W = 1.0; }
    else pair_weights(s, p->r_in, p->r_out, K, W);
}

/* O2 with classes: soft and complementary hard acceleration and potential by direct sum (Eq. 5-8 with L287) */
void p3t_oracle_direct_classes(int64_t n, const double *m, const double *q, const uint8_t *cls, const double *tab,
                               int64_t ns, const int64_t *subset,
                               double *acc_soft, double *pot_soft, double *acc_hard, double *pot_hard)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ns; ++k) {
        int64_t i = subset ? subset[k] : k;
        nsum as[3] = {{0, 0}, {0, 0}, {0, 0}}, ah[3] = {{0, 0}, {0, 0}, {0, 0}};
        nsum ps = {0, 0}, ph = {0, 0};
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            pairprm p = pair_of(tab, cls, i, j);
            double d[3] = { q[3 * i] - q[3 * j], q[3 * i + 1] - q[3 * j + 1], q[3 * i + 2] - q[3 * j + 2] };
            double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + p.eps2;
            double s = sqrt(s2), K, W;
            pair_weights_cls(&p, s, &K, &W);
            double mr1 = m[j] / s, mr3 = mr1 / s2;
            for (int c = 0; c < 3; ++c) { nadd(&as[c], -mr3 * K * d[c]); nadd(&ah[c], -mr3 * (1.0 - K) * d[c]); }
            nadd(&ps, -mr1 * W);
            nadd(&ph, -mr1 * (1.0 - W));
        }
        if (acc_soft) for (int c = 0; c < 3; ++c) acc_soft[3 * k + c] = nval(&as[c]);
        if (pot_soft) pot_soft[k] = nval(&ps);
        if (acc_hard) for (int c = 0; c < 3; ++c) acc_hard[3 * k + c] = nval(&ah[c]);
        if (pot_hard) pot_hard[k] = nval(&ph);
    }
}

/* O3 with classes: L_i = { j != i : s_ij < h_kind(i,j) }, every pair of an unsplit kind included.  Same two-pass
 * convention and band bookkeeping as p3t_oracle_neighbours (the band is around the pair's own h). */
int64_t p3t_oracle_neighbours_classes(int64_t n, const double *q, const uint8_t *cls, const double *tab,
                                      int64_t ns, const int64_t *subset,
                                      int64_t *count, const int64_t *offset, int32_t *list,
                                      double band, int64_t *band_pairs, int64_t band_cap)
{
    int64_t nband = 0;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ns; ++k) {
        int64_t i = subset ? subset[k] : k;
        int64_t c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            pairprm p = pair_of(tab, cls, i, j);
            double dx = q[3 * i] - q[3 * j], dy = q[3 * i + 1] - q[3 * j + 1], dz = q[3 * i + 2] - q[3 * j + 2];
            double s = sqrt(dx * dx + dy * dy + dz * dz + p.eps2);
            if (p.unsplit || s < p.h) {
                if (list) list[offset[k] + c] = (int32_t)j;
                ++c;
            }
            if (!p.unsplit && band > 0.0 && fabs(s / p.h - 1.0) < band) {
                int64_t slot;
#pragma omp atomic capture
                slot = nband++;
                if (band_pairs && slot < band_cap) { band_pairs[2 * slot] = k; band_pairs[2 * slot + 1] = j; }
            }
        }
        if (count) count[k] = c;
    }
    return nband;
}

/* O6 with classes: hard acceleration, jerk and potential over ALL j != i with the pair's own numbers; an unsplit
 * pair contributes the whole (eps_kind-softened) Newtonian term at every separation (1 - K = 1, dK/ds = 0). */
void p3t_oracle_hard_classes(int64_t n, const double *m, const double *q, const double *v, const uint8_t *cls,
                             const double *tab, int64_t ns, const int64_t *subset,
                             double *acc, double *jerk, double *pot)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ns; ++k) {
        int64_t i = subset ? subset[k] : k;
        nsum a[3] = {{0, 0}, {0, 0}, {0, 0}}, jk[3] = {{0, 0}, {0, 0}, {0, 0}}, ph = {0, 0};
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            pairprm p = pair_of(tab, cls, i, j);
            double d[3], w[3];
            for (int c = 0; c < 3; ++c) { d[c] = q[3 * i + c] - q[3 * j + c]; w[c] = v[3 * i + c] - v[3 * j + c]; }
            double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + p.eps2;
            double s = sqrt(s2);
            if (!p.unsplit && s >= p.r_out) continue;
            double K, W, dKds = 0.0;
            pair_weights_cls(&p, s, &K, &W);
            if (!p.unsplit) {
                double g = p.r_in / p.r_out;
                dKds = p3t_oracle_dKdx((s / p.r_out - g) / (1.0 - g)) / (p.r_out * (1.0 - g));
            }
            double qv = d[0] * w[0] + d[1] * w[1] + d[2] * w[2];
            double mr3 = m[j] / (s2 * s);
            for (int c = 0; c < 3; ++c) {
                nadd(&a[c], -mr3 * (1.0 - K) * d[c]);
                nadd(&jk[c], -mr3 * ((1.0 - K) * (w[c] - 3.0 * qv * d[c] / s2) - dKds * (qv / s) * d[c]));
            }
            nadd(&ph, -(m[j] / s) * (1.0 - W));
        }
        for (int c = 0; c < 3; ++c) {
            if (acc) acc[3 * k + c] = nval(&a[c]);
            if (jerk) jerk[3 * k + c] = nval(&jk[c]);
        }
        if (pot) pot[k] = nval(&ph);
    }
}

/*
 * O4 with classes.  A cell may stand for its bodies only if every one of them is a plain Newtonian partner (K = W = 1)
 * of every body of the target box, so clause 3 of R-MAC becomes: for every class ci in the box and every class cj in
 * the cell, kind (ci, cj) is split and D(B, AABB_C) >= h_kind.  The cell term (R-QUAD) uses ONE softening for all the
 * bodies of the cell: the split kinds must share their eps (the paper's runs do, L287: "eps = 1e-4 for the
 * interactions between FS-FS and FS-SMBH"); tab[0] is used.  Leaves: O8 direct terms and list test.
 */
typedef struct {
    walk_state w;
    const uint8_t *cls; const double *tab; const uint8_t *node_mask;
    int box_mask;
} walk_state_cls;

static void walk_rec_cls(walk_state_cls *wc, int32_t id)
{
    walk_state *w = &wc->w;
    const onode *nd = &w->t->node[id];
    if (nd->count == 0) return;
    int accept = 0;
    if (w->theta > 0.0) {
        double delta = sqrt((nd->c[0] - nd->g[0]) * (nd->c[0] - nd->g[0]) +
                            (nd->c[1] - nd->g[1]) * (nd->c[1] - nd->g[1]) +
                            (nd->c[2] - nd->g[2]) * (nd->c[2] - nd->g[2]));
        double rc = nd->side / w->theta + delta;
        double d2 = box_point_dist2(w->bmin, w->bmax, nd->c);
        double D2 = box_box_dist2(w->bmin, w->bmax, nd->bmin, nd->bmax);
        accept = d2 > rc * rc;
        for (int ci = 0; ci < 2 && accept; ++ci)
            for (int cj = 0; cj < 2 && accept; ++cj) {
                if (!((wc->box_mask >> ci) & 1) || !((wc->node_mask[id] >> cj) & 1)) continue;
                const double *t = wc->tab + 4 * (ci + cj);
                if (isinf(t[2]) || !(D2 >= t[3] * t[3])) accept = 0;
            }
    }
    if (accept) {
        double R[3] = { w->x[0] - nd->c[0], w->x[1] - nd->c[1], w->x[2] - nd->c[2] };
        double s2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2] + wc->tab[0] * wc->tab[0];
        double s = sqrt(s2), s3 = s * s2, s5 = s3 * s2, s7 = s5 * s2;
        const double *Q = nd->Q;
        double phi = -nd->M / s;
        double a[3] = { -nd->M * R[0] / s3, -nd->M * R[1] / s3, -nd->M * R[2] / s3 };
        if (w->use_quad) {
            double QR[3] = { Q[0] * R[0] + Q[3] * R[1] + Q[4] * R[2],
                             Q[3] * R[0] + Q[1] * R[1] + Q[5] * R[2],
                             Q[4] * R[0] + Q[5] * R[1] + Q[2] * R[2] };
            double RQR = R[0] * QR[0] + R[1] * QR[1] + R[2] * QR[2];
            double trQ = Q[0] + Q[1] + Q[2];
            phi += -0.5 * (3.0 * RQR / s5 - trQ / s3);
            for (int d = 0; d < 3; ++d)
                a[d] += 3.0 * QR[d] / s5 - 7.5 * RQR * R[d] / s7 + 1.5 * trQ * R[d] / s5;
        }
        for (int d = 0; d < 3; ++d) nadd(&w->a[d], a[d]);
        nadd(&w->phi, phi);
        w->n_pc++;
        return;
    }
    if (nd->leaf) {
        for (int32_t k = 0; k < nd->count; ++k) {
            int64_t j = w->t->perm[nd->first + k];
            if (j == w->i) continue;
            pairprm p = pair_of(wc->tab, wc->cls, w->i, j);
            double d[3] = { w->x[0] - w->t->q[3 * j], w->x[1] - w->t->q[3 * j + 1], w->x[2] - w->t->q[3 * j + 2] };
            double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + p.eps2;
            double s = sqrt(s2), K, W;
            pair_weights_cls(&p, s, &K, &W);
            double mr1 = w->t->m[j] / s, mr3 = mr1 / s2;
            for (int c = 0; c < 3; ++c) nadd(&w->a[c], -mr3 * K * d[c]);
            nadd(&w->phi, -mr1 * W);
            w->n_pp++;
            if (p.unsplit || s < p.h) {
                if (w->nbr && w->nbr_n < w->nbr_cap) w->nbr[w->nbr_n] = (int32_t)j;
                w->nbr_n++;
            }
        }
        return;
    }
    for (int o = 0; o < 8; ++o)
        if (nd->child[o] >= 0) walk_rec_cls(wc, nd->child[o]);
}

/* Same calling convention as p3t_oracle_tree_walk; box_mask[k] (NULL: the target's own class) is the set of classes,
 * bit 0 = FS, bit 1 = BH, present in the box of target k. */
void p3t_oracle_tree_walk_classes(const void *tree, const uint8_t *cls, const double *tab, double theta,
                                  int use_quad, int64_t ns, const int64_t *subset, const double *box, const uint8_t *box_mask,
                                  double *acc, double *pot, int64_t *counts,
                                  int32_t *nbr, int64_t nbr_stride, int64_t *nbr_count)
{
    const otree *t = (const otree *)tree;
    uint8_t *mask = (uint8_t *)calloc((size_t)t->nnode, 1);
    for (int64_t id = 0; id < t->nnode; ++id)
        for (int32_t k = 0; k < t->node[id].count; ++k) mask[id] |= (uint8_t)(1u << cls[t->perm[t->node[id].first + k]]);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t k = 0; k < ns; ++k) {
        walk_state_cls wc;
        memset(&wc, 0, sizeof wc);
        walk_state *w = &wc.w;
        w->t = t; w->i = subset ? subset[k] : k;
        for (int d = 0; d < 3; ++d) {
            w->x[d] = t->q[3 * w->i + d];
            w->bmin[d] = box ? box[6 * k + d] : w->x[d];
            w->bmax[d] = box ? box[6 * k + 3 + d] : w->x[d];
        }
        w->theta = theta; w->use_quad = use_quad;
        w->nbr = nbr ? nbr + k * nbr_stride : NULL; w->nbr_cap = nbr_stride;
        wc.cls = cls; wc.tab = tab; wc.node_mask = mask;
        wc.box_mask = box_mask ? box_mask[k] : (1 << cls[w->i]);
        walk_rec_cls(&wc, 0);
        if (acc) for (int d = 0; d < 3; ++d) acc[3 * k + d] = nval(&w->a[d]);
        if (pot) pot[k] = nval(&w->phi);
        if (counts) { counts[2 * k] = w->n_pp; counts[2 * k + 1] = w->n_pc; }
        if (nbr_count) nbr_count[k] = w->nbr_n;
        if (w->nbr && w->nbr_n > 1)
            qsort(w->nbr, (size_t)(w->nbr_n < w->nbr_cap ? w->nbr_n : w->nbr_cap), sizeof(int32_t), cmp_i32);
    }
    free(mask);
}

/*
 * O7 with classes: one soft step under H_hard with the pair kinds of O8 (L287).  The force on i over its list is Eq. 7
 * with the kind's own softening and cutoff radii; a pair of an unsplit kind contributes the whole Newtonian term
 * (1 - K = 1, dK/ds = 0) at every separation -- "the force between SMBHs is integrated with the pure Hermite scheme".
 * The accuracy parameters are per CLASS of the integrated particle: eta[c], eta_s[c], a0[c] (L287: eta_FS = 0.1,
 * eta_BH = 0.03; a0 = alpha m / r_cut^2 of Eq. 19 differs with the mass and the cutoff radius).  Everything else --
 * ticks, block steps, predictor, corrector, the order of the operations -- is O7's, restated here so that O7 itself
 * stays untouched; with all classes 0 the result equals O7's bit for bit (pinned).
 */
static void o7c_force(int64_t i, const double *m, const double *xp, const double *vp,
                      const int64_t *offset, const int32_t *list, const uint8_t *cls, const double *tab,
                      double *a, double *a1)
{
    for (int c = 0; c < 3; ++c) a[c] = a1[c] = 0.0;
    for (int64_t e = offset[i]; e < offset[i + 1]; ++e) {
        int64_t j = list[e];
        pairprm p = pair_of(tab, cls, i, j);
        const double *xj = xp + 3 * (e - offset[i] + 1), *vj = vp + 3 * (e - offset[i] + 1);
        double d[3], w[3];
        for (int c = 0; c < 3; ++c) { d[c] = xp[c] - xj[c]; w[c] = vp[c] - vj[c]; }
        double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + p.eps2;
        double s = sqrt(s2);
        if (!p.unsplit && s >= p.r_out) continue;
        double K = 0.0, W, dKds = 0.0;
        if (!p.unsplit) {
            const double g = p.r_in / p.r_out;
            pair_weights(s, p.r_in, p.r_out, &K, &W);
            dKds = p3t_oracle_dKdx((s / p.r_out - g) / (1.0 - g)) / (p.r_out * (1.0 - g));
        }
        double qv = d[0] * w[0] + d[1] * w[1] + d[2] * w[2];
        double mr3 = m[j] / (s2 * s);
        for (int c = 0; c < 3; ++c) {
            a[c] += -mr3 * (1.0 - K) * d[c];
            a1[c] += -mr3 * ((1.0 - K) * (w[c] - 3.0 * qv * d[c] / s2) - dKds * (qv / s) * d[c]);
        }
    }
}

int64_t p3t_oracle_hermite_classes(int64_t n, const double *m, double *q, double *v, const uint8_t *cls, const double *tab,
                                   const int64_t *offset, const int32_t *list,
                                   double T, int log2_div, const double *eta, const double *eta_s, const double *a0,
                                   int64_t max_blocks, int64_t *nstep, int64_t *floor_hits)
{
    const int64_t total = (int64_t)1 << O7_TICK_BITS, max_ticks = total >> log2_div;
    const double tick = T / (double)total;
    int64_t *t = calloc((size_t)n, sizeof *t), *dt = calloc((size_t)n, sizeof *dt);
    double *a = calloc((size_t)3 * n, sizeof *a), *a1 = calloc((size_t)3 * n, sizeof *a1);
    double *an = calloc((size_t)3 * n, sizeof *an), *a1n = calloc((size_t)3 * n, sizeof *a1n);
    int64_t maxl = 0, nblocks = 0;
    if (floor_hits) *floor_hits = 0;
    for (int64_t i = 0; i < n; ++i) if (offset[i + 1] - offset[i] > maxl) maxl = offset[i + 1] - offset[i];
    double *xp = malloc((size_t)3 * (maxl + 1) * sizeof *xp), *vp = malloc((size_t)3 * (maxl + 1) * sizeof *vp);

    for (int64_t i = 0; i < n; ++i) {
        if (nstep) nstep[i] = 0;
        if (offset[i + 1] == offset[i]) continue;
        for (int c = 0; c < 3; ++c) { xp[c] = q[3 * i + c]; vp[c] = v[3 * i + c]; }
        for (int64_t e = offset[i]; e < offset[i + 1]; ++e)
            for (int c = 0; c < 3; ++c) {
                xp[3 * (e - offset[i] + 1) + c] = q[3 * (int64_t)list[e] + c];
                vp[3 * (e - offset[i] + 1) + c] = v[3 * (int64_t)list[e] + c];
            }
        o7c_force(i, m, xp, vp, offset, list, cls, tab, a + 3 * i, a1 + 3 * i);
        double na = o7_norm(a + 3 * i), n1 = o7_norm(a1 + 3 * i), A0 = a0[cls[i]];
        double crit = n1 > 0.0 ? eta_s[cls[i]] * sqrt((na * na + A0 * A0) / (n1 * n1)) : INFINITY;
        dt[i] = o7_quantise(crit, tick, max_ticks, 0, floor_hits);
    }
    for (;;) {
        int64_t tn = INT64_MAX;
        for (int64_t i = 0; i < n; ++i)
            if (offset[i + 1] > offset[i] && t[i] < total && t[i] + dt[i] < tn) tn = t[i] + dt[i];
        if (tn == INT64_MAX) break;
        if (++nblocks > max_blocks) { nblocks = -1; break; }
        for (int64_t i = 0; i < n; ++i) {
            if (offset[i + 1] == offset[i] || t[i] + dt[i] != tn) continue;
            for (int64_t k = 0; k <= offset[i + 1] - offset[i]; ++k) {
                int64_t j = k ? (int64_t)list[offset[i] + k - 1] : i;
                double h = (double)(tn - t[j]) * tick;
                for (int c = 0; c < 3; ++c) {
                    double A = a[3 * j + c], J = a1[3 * j + c];
                    xp[3 * k + c] = q[3 * j + c] + h * (v[3 * j + c] + h * (A / 2.0 + h * (J / 6.0)));
                    vp[3 * k + c] = v[3 * j + c] + h * (A + h * (J / 2.0));
                }
            }
            o7c_force(i, m, xp, vp, offset, list, cls, tab, an + 3 * i, a1n + 3 * i);
        }
        for (int64_t i = 0; i < n; ++i) {
            if (offset[i + 1] == offset[i] || t[i] + dt[i] != tn) continue;
            double h = (double)dt[i] * tick, a2[3], a3[3], a2e[3];
            for (int c = 0; c < 3; ++c) {
                double A = a[3 * i + c], J = a1[3 * i + c], An = an[3 * i + c], Jn = a1n[3 * i + c];
                a2[c] = (-6.0 * (A - An) - h * (4.0 * J + 2.0 * Jn)) / (h * h);
                a3[c] = (12.0 * (A - An) + 6.0 * h * (J + Jn)) / (h * h * h);
                double x_p = q[3 * i + c] + h * (v[3 * i + c] + h * (A / 2.0 + h * (J / 6.0)));
                double v_p = v[3 * i + c] + h * (A + h * (J / 2.0));
                q[3 * i + c] = x_p + h * h * h * h * (a2[c] / 24.0 + h * a3[c] / 120.0);
                v[3 * i + c] = v_p + h * h * h * (a2[c] / 6.0 + h * a3[c] / 24.0);
                a2e[c] = a2[c] + h * a3[c];
                a[3 * i + c] = An; a1[3 * i + c] = Jn;
            }
            t[i] = tn;
            if (nstep) ++nstep[i];
            double na = o7_norm(a + 3 * i), n1 = o7_norm(a1 + 3 * i), n2 = o7_norm(a2e), n3 = o7_norm(a3), A0 = a0[cls[i]];
            double den = n1 * n3 + n2 * n2;
            double crit = den > 0.0 ? eta[cls[i]] * sqrt((sqrt(na * na + A0 * A0) * n2 + n1 * n1) / den) : INFINITY;
            dt[i] = o7_quantise(crit, tick, max_ticks, tn, floor_hits);
        }
    }
    for (int64_t i = 0; i < n && nblocks >= 0; ++i)
        if (offset[i + 1] == offset[i])
            for (int c = 0; c < 3; ++c) q[3 * i + c] += T * v[3 * i + c];
    free(t); free(dt); free(a); free(a1); free(an); free(a1n); free(xp); free(vp);
    return nblocks;
}

int p3t_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
