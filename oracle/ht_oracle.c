/*
 * ht_oracle.c -- CPU ORACLE for the Hough-Transform track finder of Rinaldi et al.,
 * "GPGPU for track finding in High Energy Physics" (arXiv:1507.03074; /root/reference/PAPER.md).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.  It shares no code with the CUDA
 * library (paper_1507_03074_b200/csrc): no headers, helpers, tables or constants.
 *
 * It is the plain definition, single-threaded, in the paper's order:
 *   - fill  : PAPER.md:25 (section 2): for every hit, every circle x^2+y^2-2Ax-2By=0 through the hit
 *             and the origin; "for each A, the corresponding B is evaluated";
 *             the M_H(A,B,theta,phi) element is "incremented by one".
 *   - peaks : "elements above a given threshold ... local maxima search";
 *             PAPER.md:43 "compares one M_H element to its neighbours and, if the biggest, it is stored".
 * Where the paper is silent the readings R1-R16 of /root/repo/SPEC.md apply (listed in DESIGN.md).
 *
 * Precision: the paper does not fix one.  Floating point here DECIDES INTEGERS (bin indices), so both
 * sides take those decisions in the kernel's precision: IEEE binary32, one rounding per operation,
 * no FMA contraction.  Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math (x86-64 => SSE2 scalar).
 *
 * Pins (tests/test_oracle_*.py, all independent of this file's arithmetic): circle equation in double
 * for every vote (P1), noiseless 12-layer track => one cell with 12 (P2), vote conservation (P3),
 * cell-centric brute force in double with atan2 binning on tiny binnings (P4), single-hit geometry (P5),
 * mirror symmetry (P6), permutation/batching invariance (P7), hand-built peak matrices (P8),
 * peak-set invariants (P9), table binning vs atan2 (P10), closed-form in-range fraction; track read-out: the
 * truth circle of a noiseless track (P11), polar identities and special cells (P12); ridge merging: connected-component
 * labelling of a library routine on a doubled grid (P13), hand-built peak layouts (P14), partition invariants (P15); truth
 * matching: noiseless tracks through generator, fill, peaks and merge (P16), a sector-split soft track (P17), hand-built
 * lists (P18), invariants and a brute force in polar coordinates (P19).
 * Parity unpinned by the paper (definitions fixed by SPEC.md only): R2/R4 angle definition and
 * ranges, R5 bin centre, R10 neighbourhood, R11 >= vs >, R12 tie rule, R17 quadrant of phi, R19 (the merge rule itself
 * is this build's stand-in for the paper's unexplained step from local maxima to tracks), R20 (the matching rule: the
 * paper's own comparison is against a chi^2 fit on its dataset, both unavailable).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t n_theta, n_phi, n_a, n_b;
    float a_min, a_max, b_min, b_max;
    float theta_min, theta_max, phi_min, phi_max;
} oracle_binning;

typedef struct { uint32_t event, cell, count; } oracle_peak;

#define ORACLE_PI 3.14159265358979323846

static double cot_d(double t) { return cos(t) / sin(t); }

/* SPEC.md section 1: "diamond" pseudo-angle of an edge, evaluated in double. */
static double pseudo_d(double phi)
{
    double c = cos(phi), s = sin(phi);
    double m = fabs(c) + fabs(s);
    return (s >= 0.0) ? 1.0 - c / m : 3.0 + c / m;
}

static int binning_ok(const oracle_binning *g)
{
    if (!g) return 0;
    if (g->n_theta < 1 || g->n_phi < 1 || g->n_a < 1 || g->n_b < 1) return 0;
    if (!(g->a_min < g->a_max) || !(g->b_min < g->b_max)) return 0;
    if (!(g->theta_min < g->theta_max) || !(g->phi_min < g->phi_max)) return 0;
    if (!isfinite(g->a_min) || !isfinite(g->a_max) || !isfinite(g->b_min) || !isfinite(g->b_max)) return 0;
    return 1;
}

/*
 * SPEC.md section 1.  two_a[NA]; t_theta[Ntheta+1] (index 0 and Ntheta = outer bounds);
 * p_phi[Nphi+1] (same); d_ab[2] = {dA, dB}.
 */
int oracle_tables(const oracle_binning *g, float *two_a, float *t_theta, float *p_phi, float *d_ab)
{
    if (!binning_ok(g)) return -1;
    float dA = (g->a_max - g->a_min) / (float)g->n_a;
    float dB = (g->b_max - g->b_min) / (float)g->n_b;
    d_ab[0] = dA;
    d_ab[1] = dB;
    for (int i = 0; i < g->n_a; ++i) {
        float fi = (float)i + 0.5f;
        float ac = g->a_min + fi * dA;          /* bin centre, R5 */
        two_a[i] = 2.0f * ac;
    }
    int th_full_hi = g->theta_max >= (float)ORACLE_PI;
    int ph_full_hi = g->phi_max >= (float)(2.0 * ORACLE_PI);
    double thlo = (double)g->theta_min, thhi = th_full_hi ? ORACLE_PI : (double)g->theta_max;
    double phlo = (double)g->phi_min, phhi = ph_full_hi ? 2.0 * ORACLE_PI : (double)g->phi_max;
    t_theta[0] = (g->theta_min <= 0.0f) ? INFINITY : (float)cot_d(thlo);
    for (int k = 1; k < g->n_theta; ++k) {
        double th = thlo + ((thhi - thlo) * (double)k) / (double)g->n_theta;
        t_theta[k] = (float)cot_d(th);
    }
    t_theta[g->n_theta] = th_full_hi ? -INFINITY : (float)cot_d(thhi);
    p_phi[0] = (g->phi_min <= 0.0f) ? 0.0f : (float)pseudo_d(phlo);
    for (int k = 1; k < g->n_phi; ++k) {
        double ph = phlo + ((phhi - phlo) * (double)k) / (double)g->n_phi;
        p_phi[k] = (float)pseudo_d(ph);
    }
    p_phi[g->n_phi] = ph_full_hi ? 4.0f : (float)pseudo_d(phhi);
    return 0;
}

typedef struct {
    const oracle_binning *g;
    float *two_a, *t_theta, *p_phi;
    float dA, dB;
} tables;

static int tables_make(tables *t, const oracle_binning *g)
{
    memset(t, 0, sizeof *t);
    t->g = g;
    t->two_a = (float *)malloc(sizeof(float) * (size_t)g->n_a);
    t->t_theta = (float *)malloc(sizeof(float) * (size_t)(g->n_theta + 1));
    t->p_phi = (float *)malloc(sizeof(float) * (size_t)(g->n_phi + 1));
    float d[2];
    if (!t->two_a || !t->t_theta || !t->p_phi || oracle_tables(g, t->two_a, t->t_theta, t->p_phi, d) != 0) {
        free(t->two_a); free(t->t_theta); free(t->p_phi);
        return -1;
    }
    t->dA = d[0];
    t->dB = d[1];
    return 0;
}

static void tables_free(tables *t) { free(t->two_a); free(t->t_theta); free(t->p_phi); }

/* SPEC.md section 2, first half: the (theta,phi) plane of a hit, or -1 (R2, R3, R4, R8). */
static int32_t hit_plane(const tables *t, float x, float y, float z)
{
    const oracle_binning *g = t->g;
    float r2 = x * x + y * y;
    float q = z / sqrtf(r2);
    if (!(q <= t->t_theta[0] && q > t->t_theta[g->n_theta])) return -1;
    int it = 0;
    for (int k = 1; k < g->n_theta; ++k)
        if (q <= t->t_theta[k]) ++it;
    float d = fabsf(x) + fabsf(y);
    float u = x / d;
    float p = (y >= 0.0f) ? (1.0f - u) : (3.0f + u);
    if (!(p >= t->p_phi[0] && p < t->p_phi[g->n_phi])) return -1;
    int ip = 0;
    for (int k = 1; k < g->n_phi; ++k)
        if (p >= t->p_phi[k]) ++ip;
    return (int32_t)(it * g->n_phi + ip);
}

/* SPEC.md section 2, second half: the B bin voted by hit (x,y) in A row i, or -1 (R5, R6, R7, R8). */
static int32_t vote_bin(const tables *t, float x, float y, int i)
{
    float r2 = x * x + y * y;
    float den = 2.0f * y;
    float prod = t->two_a[i] * x;
    float num = r2 - prod;
    float B = num / den;                         /* B = (x^2+y^2-2Ax)/(2y) */
    float s = B - t->g->b_min;
    float tt = s / t->dB;
    if (tt >= 0.0f && tt < (float)t->g->n_b) return (int32_t)tt;
    return -1;
}

/*
 * Fill the vote matrix of ONE event.  M (cells uint32) is zeroed here.  Returns the number of votes
 * cast (-1 on bad arguments).  PAPER.md:25, 39-43.
 */
int64_t oracle_fill(const oracle_binning *g, const float *x, const float *y, const float *z, int64_t n_hits,
                    uint32_t *M)
{
    tables t;
    if (!binning_ok(g) || n_hits < 0 || !M || tables_make(&t, g) != 0) return -1;
    size_t cells = (size_t)g->n_theta * (size_t)g->n_phi * (size_t)g->n_a * (size_t)g->n_b;
    memset(M, 0, cells * sizeof(uint32_t));
    int64_t votes = 0;
    for (int64_t h = 0; h < n_hits; ++h) {
        int32_t plane = hit_plane(&t, x[h], y[h], z[h]);
        if (plane < 0) continue;
        for (int i = 0; i < g->n_a; ++i) {
            int32_t b = vote_bin(&t, x[h], y[h], i);
            if (b < 0) continue;
            size_t cell = ((size_t)plane * (size_t)g->n_a + (size_t)i) * (size_t)g->n_b + (size_t)b;
            M[cell] += 1u;                       /* "incremented by one" */
            ++votes;
        }
    }
    tables_free(&t);
    return votes;
}

/*
 * The same decisions as oracle_fill, without the matrix: plane[h] (or -1) and bins[h*NA + i] (or -1).
 * Exists so that tests can check every single vote against the circle equation (pin P1) and count
 * votes without a matrix (pin P3).
 */
int oracle_votes(const oracle_binning *g, const float *x, const float *y, const float *z, int64_t n_hits,
                 int32_t *plane, int32_t *bins)
{
    tables t;
    if (!binning_ok(g) || n_hits < 0 || tables_make(&t, g) != 0) return -1;
    for (int64_t h = 0; h < n_hits; ++h) {
        plane[h] = hit_plane(&t, x[h], y[h], z[h]);
        for (int i = 0; i < g->n_a; ++i)
            bins[h * (int64_t)g->n_a + i] = (plane[h] < 0) ? -1 : vote_bin(&t, x[h], y[h], i);
    }
    tables_free(&t);
    return 0;
}

/*
 * Peak search over ONE event's matrix (SPEC.md section 3).  Emits peaks in increasing
 * cell order; writes at most `capacity`; returns the number found (-1 on bad arguments).
 */
int64_t oracle_peaks(const oracle_binning *g, const uint32_t *M, uint32_t threshold, uint32_t event,
                     oracle_peak *out, int64_t capacity)
{
    if (!binning_ok(g) || !M || threshold < 1u || capacity < 0) return -1;
    const int64_t NA = g->n_a, NB = g->n_b, P = (int64_t)g->n_theta * g->n_phi;
    int64_t found = 0;
    for (int64_t p = 0; p < P; ++p) {
        const uint32_t *plane = M + (size_t)p * (size_t)NA * (size_t)NB;
        for (int64_t a = 0; a < NA; ++a) {
            for (int64_t b = 0; b < NB; ++b) {
                uint32_t c = plane[a * NB + b];
                if (c < threshold) continue;                     /* R11 */
                int is_peak = 1;
                for (int da = -1; da <= 1 && is_peak; ++da) {
                    for (int db = -1; db <= 1; ++db) {
                        if (da == 0 && db == 0) continue;
                        int64_t a2 = a + da, b2 = b + db;
                        if (a2 < 0 || a2 >= NA || b2 < 0 || b2 >= NB) continue;   /* R10 */
                        uint32_t nb = plane[a2 * NB + b2];
                        int earlier = (da < 0) || (da == 0 && db < 0);
                        if (earlier ? (nb >= c) : (nb > c)) { is_peak = 0; break; }  /* R12 */
                    }
                }
                if (!is_peak) continue;
                if (found < capacity) {
                    out[found].event = event;
                    out[found].cell = (uint32_t)((p * NA + a) * NB + b);
                    out[found].count = c;
                }
                ++found;
            }
        }
    }
    return found;
}

/*
 * Track read-out of a peak (SPEC.md section 4; "rho = sqrt(A^2 + B^2) and phi = tan^-1(B/A)"):
 * (A, B) = centre of the peak's (A, B) cell = centre of the track's circle (the circle through the
 * origin with centre (A, B) is x^2+y^2-2Ax-2By=0), so rho is the circle's radius and phi the azimuth of its
 * centre.  Reading R17: tan^-1(B/A) is taken quadrant-aware (atan2), in (-pi, pi]; R18: (A, B) are the bin
 * centres of R5, evaluated in binary32 exactly as the row values of the fill (they are inputs of the method,
 * not results); rho and phi are then the PLAIN DEFINITION in double precision -- the CUDA path computes them
 * in binary32 and is compared within a tolerance, no integer depends on them.
 * Returns 0, or -1 on bad arguments.  Pins: P11 (truth circle of a noiseless track), P12 (identities).
 */
int oracle_tracks(const oracle_binning *g, const oracle_peak *peaks, int64_t n, double *rho, double *phi)
{
    if (!binning_ok(g) || n < 0 || (n > 0 && (!peaks || !rho || !phi))) return -1;
    const float dA = (g->a_max - g->a_min) / (float)g->n_a;
    const float dB = (g->b_max - g->b_min) / (float)g->n_b;
    const uint64_t cells = (uint64_t)g->n_theta * g->n_phi * g->n_a * g->n_b;
    for (int64_t k = 0; k < n; ++k) {
        if (peaks[k].cell >= cells) return -1;
        const uint32_t ib = peaks[k].cell % (uint32_t)g->n_b;
        const uint32_t ia = (peaks[k].cell / (uint32_t)g->n_b) % (uint32_t)g->n_a;
        const float fa = (float)ia + 0.5f, fb = (float)ib + 0.5f;
        const float pa = fa * dA, pb = fb * dB;
        const float A = g->a_min + pa, B = g->b_min + pb;          /* bin centres (R5, R18) */
        rho[k] = sqrt((double)A * (double)A + (double)B * (double)B);
        phi[k] = atan2((double)B, (double)A);
    }
    return 0;
}

/*
 * Ridge merging of a peak list (SPEC.md section 5, reading R19; SURVEY.md section 8(f) f3 "merging ridge peaks").
 * PAPER.md:25 goes from "local maxima" straight to "real tracks"; a stiff track's vote lines are nearly parallel, so its
 * maximum is a RIDGE on which several non-adjacent cells pass the peak rule.  R19: two peaks of the same event and the
 * same (theta,phi) plane are LINKED when their cells are at Chebyshev distance <= window in (a, b); a track candidate is
 * a connected component of the link graph; its representative is the member with the largest count, the smallest cell
 * among equals.  out[k] = (event, representative cell, its count, members, rho, phi of the representative as in
 * oracle_tracks), sorted by (event, cell).  Plain definition: every pair is tested, textbook union-find.
 * Returns the number of components (-1 on bad arguments); writes at most `capacity`.
 */
typedef struct { uint32_t event, cell, count, n_peaks; double rho, phi; } oracle_merged;

static int64_t uf_find(int64_t *parent, int64_t i)
{
    while (parent[i] != i) i = parent[i];
    return i;
}

static int merged_less(const oracle_merged *a, const oracle_merged *b)
{
    return a->event < b->event || (a->event == b->event && a->cell < b->cell);
}

int64_t oracle_merge_ridges(const oracle_binning *g, const oracle_peak *peaks, int64_t n, uint32_t window,
                            oracle_merged *out, int64_t capacity)
{
    if (!binning_ok(g) || n < 0 || capacity < 0 || (n > 0 && !peaks)) return -1;
    const int64_t NA = g->n_a, NB = g->n_b;
    const uint64_t cells = (uint64_t)g->n_theta * g->n_phi * g->n_a * g->n_b;
    for (int64_t i = 0; i < n; ++i)
        if (peaks[i].cell >= cells) return -1;
    int64_t *parent = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n + 1));
    if (!parent) return -1;
    for (int64_t i = 0; i < n; ++i) parent[i] = i;
    for (int64_t i = 0; i < n; ++i) {
        const int64_t bi = peaks[i].cell % NB, ai = (peaks[i].cell / NB) % NA, pi = peaks[i].cell / (NB * NA);
        for (int64_t j = i + 1; j < n; ++j) {
            if (peaks[j].event != peaks[i].event) continue;
            const int64_t bj = peaks[j].cell % NB, aj = (peaks[j].cell / NB) % NA, pj = peaks[j].cell / (NB * NA);
            if (pj != pi) continue;                                  /* never across (theta,phi) planes (R10) */
            const int64_t da = ai > aj ? ai - aj : aj - ai, db = bi > bj ? bi - bj : bj - bi;
            if ((da > db ? da : db) > (int64_t)window) continue;    /* Chebyshev distance */
            const int64_t ri = uf_find(parent, i), rj = uf_find(parent, j);
            if (ri != rj) parent[ri] = rj;
        }
    }
    int64_t found = 0;
    oracle_merged *all = (oracle_merged *)malloc(sizeof(oracle_merged) * (size_t)(n + 1));
    if (!all) { free(parent); return -1; }
    for (int64_t r = 0; r < n; ++r) {
        if (parent[r] != r) continue;                                /* one component per root */
        int64_t best = -1;
        uint32_t members = 0;
        for (int64_t i = 0; i < n; ++i) {
            if (uf_find(parent, i) != r) continue;
            ++members;
            if (best < 0 || peaks[i].count > peaks[best].count ||
                (peaks[i].count == peaks[best].count && peaks[i].cell < peaks[best].cell)) best = i;
        }
        oracle_merged m;
        m.event = peaks[best].event; m.cell = peaks[best].cell; m.count = peaks[best].count; m.n_peaks = members;
        oracle_peak one = peaks[best];
        if (oracle_tracks(g, &one, 1, &m.rho, &m.phi) != 0) { free(parent); free(all); return -1; }
        all[found++] = m;
    }
    for (int64_t i = 1; i < found; ++i) {                            /* insertion sort by (event, cell) */
        oracle_merged key = all[i];
        int64_t j = i - 1;
        while (j >= 0 && merged_less(&key, &all[j])) { all[j + 1] = all[j]; --j; }
        all[j + 1] = key;
    }
    for (int64_t i = 0; i < found && i < capacity; ++i) out[i] = all[i];
    free(parent);
    free(all);
    return found;
}

/*
 * Truth matching of track candidates (SPEC.md section 6, reading R20; SURVEY.md section 8(f) f3 "truth-matched
 * efficiency / fake rate / resolution on the synthetic events"; the stand-in for PAPER.md:29-33, Fig. 1, where "the
 * rho = sqrt(A^2+B^2) and phi = tan^-1(B/A) are shown together with the corresponding resolutions").
 * A candidate stands for the circle through the origin whose centre (A_c, B_c) is the centre of its cell (section 4);
 * a generated track IS such a circle with centre (A_t, B_t) (generator G3).  All arithmetic in binary64, one rounding
 * per operation, in the order written; no arctangent enters a decision:
 *   rho_c = sqrt(A_c*A_c + B_c*B_c), rho_t alike
 *   compatible(c, t)  <=>  same event  and  |rho_c - rho_t| <= w_rho  and  A_c*A_t + B_c*B_t >= cos_w_phi * (rho_c*rho_t)
 *   d2(c, t) = (A_c-A_t)^2 + (B_c-B_t)^2
 *   cand_match[c]  = the compatible t of smallest d2 (ties: smallest index t), or -1: the candidate is a FAKE
 *   truth_match[t] = among the c with cand_match[c] == t the one of smallest d2 (ties: smallest cell), or -1: NOT FOUND;
 *                    the other candidates matched to t are DUPLICATES
 *   residuals of a found track, with c = truth_match[t]: d_rho = rho_c - rho_t, d_phi = atan2(A_t*B_c - B_t*A_c, A_c*A_t + B_c*B_t)
 * Returns 0, or -1 on bad arguments.  Pins: P16 (noiseless tracks through generator, fill, peaks, merge: all found, no
 * fake, residuals below one cell diagonal), P17 (a soft track split by a sector edge is not found), P18 (hand-built
 * lists), P19 (invariants, and a brute force in polar coordinates away from the window edges).
 */
typedef struct { uint32_t event, pad; double a, b; } oracle_truth;
typedef struct {
    int64_t n_cand, n_truth, n_matched, n_fake, n_found, n_duplicate;
    double sum_drho, sum_drho2, sum_dphi, sum_dphi2;        /* over the found tracks */
} oracle_match_summary;

int oracle_match_truth(const oracle_binning *g, const oracle_merged *cand, int64_t n_cand, const oracle_truth *truth,
                       int64_t n_truth, double w_rho, double cos_w_phi, int32_t *cand_match, int32_t *truth_match,
                       oracle_match_summary *sum)
{
    if (!binning_ok(g) || n_cand < 0 || n_truth < 0 || !sum) return -1;
    if ((n_cand > 0 && (!cand || !cand_match)) || (n_truth > 0 && (!truth || !truth_match))) return -1;
    if (!(w_rho >= 0.0) || !(cos_w_phi >= -1.0 && cos_w_phi <= 1.0)) return -1;
    const float dA = (g->a_max - g->a_min) / (float)g->n_a;
    const float dB = (g->b_max - g->b_min) / (float)g->n_b;
    const uint64_t cells = (uint64_t)g->n_theta * g->n_phi * g->n_a * g->n_b;
    double *best_d2 = (double *)malloc(sizeof(double) * (size_t)(n_truth + 1));
    if (!best_d2) return -1;
    for (int64_t t = 0; t < n_truth; ++t) truth_match[t] = -1;
    memset(sum, 0, sizeof *sum);
    sum->n_cand = n_cand;
    sum->n_truth = n_truth;
    for (int64_t c = 0; c < n_cand; ++c) {
        if (cand[c].cell >= cells) { free(best_d2); return -1; }
        const uint32_t ib = cand[c].cell % (uint32_t)g->n_b;
        const uint32_t ia = (cand[c].cell / (uint32_t)g->n_b) % (uint32_t)g->n_a;
        const float fa = (float)ia + 0.5f, fb = (float)ib + 0.5f;
        const float pa = fa * dA, pb = fb * dB;
        const float Af = g->a_min + pa, Bf = g->b_min + pb;            /* bin centres (R5, R18), binary32 as in section 4 */
        const double Ac = (double)Af, Bc = (double)Bf;
        const double rho_c = sqrt(Ac * Ac + Bc * Bc);
        int64_t best = -1;
        double best_c = 0.0;
        for (int64_t t = 0; t < n_truth; ++t) {
            if (truth[t].event != cand[c].event) continue;
            const double At = truth[t].a, Bt = truth[t].b;
            const double rho_t = sqrt(At * At + Bt * Bt);
            const double dr = rho_c - rho_t;
            if (!(fabs(dr) <= w_rho)) continue;
            const double dot = Ac * At + Bc * Bt;
            if (!(dot >= cos_w_phi * (rho_c * rho_t))) continue;
            const double ea = Ac - At, eb = Bc - Bt;
            const double d2 = ea * ea + eb * eb;
            if (best < 0 || d2 < best_c) { best = t; best_c = d2; }
        }
        cand_match[c] = (int32_t)best;
        if (best < 0) { ++sum->n_fake; continue; }
        ++sum->n_matched;
        const int32_t cur = truth_match[best];
        if (cur < 0 || best_c < best_d2[best] || (best_c == best_d2[best] && cand[c].cell < cand[cur].cell)) {
            truth_match[best] = (int32_t)c;
            best_d2[best] = best_c;
        }
    }
    for (int64_t t = 0; t < n_truth; ++t) {
        const int32_t c = truth_match[t];
        if (c < 0) continue;
        ++sum->n_found;
        const uint32_t ib = cand[c].cell % (uint32_t)g->n_b;
        const uint32_t ia = (cand[c].cell / (uint32_t)g->n_b) % (uint32_t)g->n_a;
        const float fa = (float)ia + 0.5f, fb = (float)ib + 0.5f;
        const float pa = fa * dA, pb = fb * dB;
        const float Af = g->a_min + pa, Bf = g->b_min + pb;
        const double Ac = (double)Af, Bc = (double)Bf, At = truth[t].a, Bt = truth[t].b;
        const double dr = sqrt(Ac * Ac + Bc * Bc) - sqrt(At * At + Bt * Bt);
        const double dp = atan2(At * Bc - Bt * Ac, Ac * At + Bc * Bt);
        sum->sum_drho += dr; sum->sum_drho2 += dr * dr;
        sum->sum_dphi += dp; sum->sum_dphi2 += dp * dp;
    }
    sum->n_duplicate = sum->n_matched - sum->n_found;
    free(best_d2);
    return 0;
}
