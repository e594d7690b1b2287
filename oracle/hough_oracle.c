/* Plain single-threaded C oracle of the Hough track-finding hot path.
 *
 * TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.  Built by oracle/hough_c.py with gcc; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no
 * code, header, table or constant generator with the CUDA path and is never linked into it.
 *
 * It is the twin of oracle/hough_def.py (pure-Python integers) for inputs too large for Python loops;
 * tests/test_oracle_pins.py checks that the two agree and pins both against closed forms, invariants,
 * library special cases and brute force.  No blocking, no SIMD, no threads: every step is the definition.
 *
 *   O1 quantise   valid <=> finite and |u|,|v| <= coord_max; u_q = rint(u 2^H) ties-to-even   (A4/A5/A14)
 *   O2 constants  F, M, C_q[t] = llround(cos(pi t / n_theta) M), S_q, O_q, W_q                (A2/A4)
 *   O3 vote       rho = phi cos(theta) + z sin(theta), Eq. 4.1; histogram with floor
 *                 binning over theta in [0,180deg); one vote per (hit, theta) L106
 *   O4 peaks      PAPER.md L94/L106 "bin with the highest number of entries", generalised to every strict
 *                 local maximum >= T under the total order (count, -index)                    (A7/A8)
 *   O5 clusters   8-connected components of the thresholded mask (keyword L29)                (A7)
 *                 theta_wrap != 0 (reading B9): O4 / O5 on the neighbourhood that continues past the theta seam,
 *                 row n_theta = row 0 with rho mirrored (Eq. 4.1: (theta + pi, rho) = (theta, -rho))
 *   O6 rank       (votes desc, index asc), keep K                                             (A11)
 *   O7 assign     PAPER.md L106 "hits that align with the straight line" -> nearest kept candidate
 *                 within the window, integer residual at the candidate's theta               (A12/A13)
 *   O8 digest     sum_b acc(b) * splitmix64(L(b)) mod 2^64
 *
 * Parity status: as in hough_def.py -- the arithmetic is pinned, the readings A2, A6-A13 are "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t n_theta, n_rho;
    double rho_min, rho_max, coord_max;
    int32_t vote_threshold;
    double assign_window;
    int32_t max_candidates;
    int32_t hit_frac_bits;
    int32_t acc_frac_bits; /* < 0: default */
    double theta_min, theta_max; /* theta window in radians; (0, 0) = the paper's [0, pi) */
    int32_t theta_wrap;          /* != 0: O4 / O5 continue past the last theta row into row 0 with rho mirrored (reading B9) */
    int32_t reserved;
} ho_params_t;

typedef struct { /* 32 bytes, the record layout the public ABI documents */
    int32_t theta_bin, rho_bin, votes, cluster_root, cluster_nbins;
    float theta, rho;
    int32_t reserved;
} ho_cand_t;

#define HO_OK 0
#define HO_EBOUND (-1) /* int32 bound of the fixed-point design violated */
#define HO_ENOMEM (-2)
#define HO_EARG (-3)

static const double HO_PI = 3.14159265358979323846;

/* theta_t = theta_min + (theta_max - theta_min) t / n_theta; a window of (0, 0) means the paper's [0, pi),
 * for which this is pi t / n_theta bit for bit (x + 0.0 == x). */
static double ho_theta(const ho_params_t* p, int t)
{
    const double lo = p->theta_min, hi = (p->theta_min == 0.0 && p->theta_max == 0.0) ? HO_PI : p->theta_max;
    return lo + (hi - lo) * t / p->n_theta;
}

static double pow2i(int e) { return ldexp(1.0, e); }

/* Every intermediate of O3 and O7 fits int32 for every valid hit: q_max (max_t |C_q| + |S_q|) + |O_q| <= 2^31 - 1 with
 * q_max = floor(coord_max 2^H + 1/2), and (n_rho + 1) 2^F <= 2^31 - 1. */
static int ho_int32_proof(const ho_params_t* p, int F)
{
    const int H = p->hit_frac_bits;
    const double d_rho = (p->rho_max - p->rho_min) / p->n_rho;
    const double M = pow2i(F - H) / d_rho;
    double max_cs = 0.0;
    for (int t = 0; t < p->n_theta; ++t) {
        const double th = ho_theta(p, t);
        const double cs = fabs((double)llround(cos(th) * M)) + fabs((double)llround(sin(th) * M));
        if (cs > max_cs) max_cs = cs;
    }
    const double qmax = floor(p->coord_max * pow2i(H) + 0.5);
    const double oq = fabs((double)llround(-p->rho_min * pow2i(F) / d_rho));
    return qmax * max_cs + oq <= 2147483647.0 && ((double)p->n_rho + 1.0) * pow2i(F) <= 2147483647.0;
}

int ho_default_frac_bits(const ho_params_t* p)
{
    double d_rho = (p->rho_max - p->rho_min) / p->n_rho;
    double a = fabs(p->rho_min), b = fabs(p->rho_max);
    double span = sqrt(2.0) * p->coord_max / d_rho + (a > b ? a : b) / d_rho + 2.0;
    int F = 24;
    if (span < (double)p->n_rho + 1.0) span = (double)p->n_rho + 1.0;  /* bin centres r 2^F + 2^(F-1), r < n_rho (O7) */
    while (F > 0 && span * pow2i(F) > 2147483647.0) --F;
    while (F > 1 && !ho_int32_proof(p, F)) --F;  /* d_rho far below the hit resolution: the closed form is not enough */
    return F;
}

/* scal = {H, F, O_q, W_q} */
int ho_constants(const ho_params_t* p, int64_t* Cq, int64_t* Sq, int64_t* scal)
{
    if (p->n_theta < 1 || p->n_rho < 1 || !(p->rho_max > p->rho_min)) return HO_EARG;
    int H = p->hit_frac_bits;
    int F = p->acc_frac_bits >= 0 ? p->acc_frac_bits : ho_default_frac_bits(p);
    double d_rho = (p->rho_max - p->rho_min) / p->n_rho;
    double M = pow2i(F - H) / d_rho;
    for (int t = 0; t < p->n_theta; ++t) {
        double th = ho_theta(p, t);
        Cq[t] = llround(cos(th) * M);
        Sq[t] = llround(sin(th) * M);
    }
    scal[0] = H;
    scal[1] = F;
    scal[2] = llround(-p->rho_min * pow2i(F) / d_rho);
    scal[3] = llround(p->assign_window * pow2i(F) / d_rho);
    return HO_OK;
}

static int quantise(const ho_params_t* p, int H, float u, float v, int64_t* uq, int64_t* vq)
{
    double ud = (double)u, vd = (double)v;
    if (!isfinite(ud) || !isfinite(vd)) return 0;
    if (fabs(ud) > p->coord_max || fabs(vd) > p->coord_max) return 0;
    *uq = (int64_t)nearbyint(ud * pow2i(H)); /* default rounding mode: ties to even */
    *vq = (int64_t)nearbyint(vd * pow2i(H));
    return 1;
}

static int64_t iabs64(int64_t x) { return x < 0 ? -x : x; }

/* floor(a / 2^F) for signed a */
static int64_t floor_shift(int64_t a, int F)
{
    int64_t d = (int64_t)1 << F;
    int64_t q = a / d;
    if ((a % d) != 0 && a < 0) --q;
    return q;
}

int ho_vote_event(const ho_params_t* p, const float* u, const float* v, int64_t n, int32_t* acc)
{
    int rc = HO_OK;
    int64_t* Cq = (int64_t*)malloc(sizeof(int64_t) * p->n_theta);
    int64_t* Sq = (int64_t*)malloc(sizeof(int64_t) * p->n_theta);
    int64_t scal[4];
    if (!Cq || !Sq) { free(Cq); free(Sq); return HO_ENOMEM; }
    if ((rc = ho_constants(p, Cq, Sq, scal)) != HO_OK) { free(Cq); free(Sq); return rc; }
    const int H = (int)scal[0], F = (int)scal[1];
    const int64_t Oq = scal[2];
    memset(acc, 0, sizeof(int32_t) * (size_t)p->n_theta * p->n_rho);
    for (int64_t i = 0; i < n; ++i) {
        int64_t uq, vq;
        if (!quantise(p, H, u[i], v[i], &uq, &vq)) continue;
        for (int t = 0; t < p->n_theta; ++t) {
            int64_t a = uq * Cq[t] + vq * Sq[t] + Oq;
            if (iabs64(uq * Cq[t]) + iabs64(vq * Sq[t]) + iabs64(Oq) > 2147483647LL) rc = HO_EBOUND;
            int64_t r = floor_shift(a, F);
            if (r >= 0 && r < p->n_rho) acc[(size_t)t * p->n_rho + r] += 1;
        }
    }
    free(Cq); free(Sq);
    return rc;
}

/* key(b) > key(n)  with key = (count, -index) */
static int key_greater(const int32_t* acc, int64_t b, int64_t n)
{
    if (acc[b] != acc[n]) return acc[b] > acc[n];
    return b < n;
}

/* Linear index of the 8-neighbour (t + dt, r + dr) of bin (t, r), or -1 if it is outside the grid.  With theta_wrap (reading
 * B9: the line (theta + pi, rho) is the line (theta, -rho), so for theta in [0, pi) and rho_min = -rho_max the row after the last
 * one is row 0 with the rho bins in reverse order) the step across the seam mirrors the rho bin: r -> n_rho - 1 - r. */
static int64_t ho_neighbour(const ho_params_t* p, int t, int r, int dt, int dr)
{
    int tt = t + dt, rr = r + dr;
    if (p->theta_wrap && tt < 0) { tt += p->n_theta; rr = p->n_rho - 1 - rr; }
    else if (p->theta_wrap && tt >= p->n_theta) { tt -= p->n_theta; rr = p->n_rho - 1 - rr; }
    if (tt < 0 || tt >= p->n_theta || rr < 0 || rr >= p->n_rho) return -1;
    return (int64_t)tt * p->n_rho + rr;
}

typedef struct { int64_t L; int32_t votes; } ho_peak_t;

static int peak_cmp(const void* x, const void* y)
{
    const ho_peak_t* a = (const ho_peak_t*)x;
    const ho_peak_t* b = (const ho_peak_t*)y;
    if (a->votes != b->votes) return a->votes > b->votes ? -1 : 1;
    return a->L < b->L ? -1 : (a->L > b->L ? 1 : 0);
}

int ho_find_clusters_event(const ho_params_t* p, const int32_t* acc, ho_cand_t* cands, int32_t* n_found)
{
    const int nt = p->n_theta, nr = p->n_rho, T = p->vote_threshold, K = p->max_candidates;
    const int64_t nb = (int64_t)nt * nr;
    if (p->theta_wrap) { /* B9 needs the paper's window, a symmetric rho range and three distinct rows around every row */
        const int default_window = (p->theta_min == 0.0 && (p->theta_max == 0.0 || p->theta_max == HO_PI));
        if (!default_window || p->rho_min != -p->rho_max || nt < 3) return HO_EARG;
    }
    /* O5: flood fill of the on-mask, 8-connectivity (no wrap unless theta_wrap) */
    int32_t* comp = (int32_t*)malloc(sizeof(int32_t) * nb);     /* component id per bin, -1 = off/unvisited */
    int64_t* stack = (int64_t*)malloc(sizeof(int64_t) * nb);
    int64_t* comp_root = (int64_t*)malloc(sizeof(int64_t) * (nb / 1 + 1));
    int32_t* comp_size = (int32_t*)malloc(sizeof(int32_t) * (nb / 1 + 1));
    ho_peak_t* pk = (ho_peak_t*)malloc(sizeof(ho_peak_t) * (nb + 1));
    if (!comp || !stack || !comp_root || !comp_size || !pk) { free(comp); free(stack); free(comp_root); free(comp_size); free(pk); return HO_ENOMEM; }
    for (int64_t b = 0; b < nb; ++b) comp[b] = -1;
    int32_t n_comp = 0;
    for (int64_t b0 = 0; b0 < nb; ++b0) {
        if (acc[b0] < T || comp[b0] >= 0) continue;
        int64_t sp = 0, root = b0;
        int32_t size = 0;
        stack[sp++] = b0;
        comp[b0] = n_comp;
        while (sp > 0) {
            int64_t b = stack[--sp];
            ++size;
            if (key_greater(acc, b, root)) root = b;
            int t = (int)(b / nr), r = (int)(b % nr);
            for (int dt = -1; dt <= 1; ++dt)
                for (int dr = -1; dr <= 1; ++dr) {
                    if (!dt && !dr) continue;
                    int64_t n = ho_neighbour(p, t, r, dt, dr);
                    if (n < 0) continue;
                    if (acc[n] >= T && comp[n] < 0) { comp[n] = n_comp; stack[sp++] = n; }
                }
        }
        comp_root[n_comp] = root;
        comp_size[n_comp] = size;
        ++n_comp;
    }
    /* O4: strict local maxima of the on-mask */
    int64_t np_ = 0;
    for (int64_t b = 0; b < nb; ++b) {
        if (acc[b] < T) continue;
        int t = (int)(b / nr), r = (int)(b % nr), is_peak = 1;
        for (int dt = -1; dt <= 1 && is_peak; ++dt)
            for (int dr = -1; dr <= 1; ++dr) {
                if (!dt && !dr) continue;
                int64_t n = ho_neighbour(p, t, r, dt, dr);
                if (n < 0 || n == b) continue;
                if (key_greater(acc, n, b)) { is_peak = 0; break; }
            }
        if (is_peak) { pk[np_].L = b; pk[np_].votes = acc[b]; ++np_; }
    }
    /* O6: rank, truncate, emit */
    qsort(pk, (size_t)np_, sizeof(ho_peak_t), peak_cmp);
    *n_found = (int32_t)np_;
    int64_t n_kept = np_ < K ? np_ : K;
    double d_rho = (p->rho_max - p->rho_min) / p->n_rho;
    for (int64_t s = 0; s < n_kept; ++s) {
        int64_t L = pk[s].L;
        int t = (int)(L / nr), r = (int)(L % nr);
        int32_t c = comp[L];
        int32_t root_slot = -1;
        for (int64_t s2 = 0; s2 <= s; ++s2)
            if (pk[s2].L == comp_root[c]) { root_slot = (int32_t)s2; break; }
        cands[s].theta_bin = t;
        cands[s].rho_bin = r;
        cands[s].votes = pk[s].votes;
        cands[s].cluster_root = root_slot;
        cands[s].cluster_nbins = comp_size[c];
        cands[s].theta = (float)ho_theta(p, t);
        cands[s].rho = (float)(p->rho_min + (r + 0.5) * d_rho);
        cands[s].reserved = 0;
    }
    free(comp); free(stack); free(comp_root); free(comp_size); free(pk);
    return HO_OK;
}

int ho_assign_event(const ho_params_t* p, const float* u, const float* v, int64_t n,
                    const ho_cand_t* cands, int32_t n_kept, int32_t* labels)
{
    int rc = HO_OK;
    int64_t* Cq = (int64_t*)malloc(sizeof(int64_t) * p->n_theta);
    int64_t* Sq = (int64_t*)malloc(sizeof(int64_t) * p->n_theta);
    int64_t scal[4];
    if (!Cq || !Sq) { free(Cq); free(Sq); return HO_ENOMEM; }
    if ((rc = ho_constants(p, Cq, Sq, scal)) != HO_OK) { free(Cq); free(Sq); return rc; }
    const int H = (int)scal[0], F = (int)scal[1];
    const int64_t Oq = scal[2], Wq = scal[3];
    const int64_t half = F >= 1 ? ((int64_t)1 << (F - 1)) : 0;
    for (int64_t i = 0; i < n; ++i) {
        int64_t uq, vq;
        labels[i] = -1;
        if (!quantise(p, H, u[i], v[i], &uq, &vq)) continue;
        int64_t best = -1;
        for (int32_t s = 0; s < n_kept; ++s) {
            int t = cands[s].theta_bin;
            int64_t a = uq * Cq[t] + vq * Sq[t] + Oq;
            int64_t e = a - ((int64_t)cands[s].rho_bin * ((int64_t)1 << F) + half);
            if (iabs64(e) > 2147483647LL) rc = HO_EBOUND;
            if (iabs64(e) <= Wq && (best < 0 || iabs64(e) < best)) { best = iabs64(e); labels[i] = s; }
        }
    }
    free(Cq); free(Sq);
    return rc;
}

static uint64_t mix64(uint64_t x)
{
    uint64_t z = x + 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

uint64_t ho_digest(const int32_t* acc, int32_t n_theta, int32_t n_rho)
{
    uint64_t d = 0;
    const int64_t nb = (int64_t)n_theta * n_rho;
    for (int64_t b = 0; b < nb; ++b)
        if (acc[b]) d += (uint64_t)(uint32_t)acc[b] * mix64((uint64_t)b);
    return d;
}

/* Whole path over a batch of events.  Nullable outputs: digest [E], acc_out [E][n_theta][n_rho],
 * cands [E][K] (with n_found [E]), labels [N].  Returns the first non-zero status. */
int ho_run_batch(const ho_params_t* p, const float* u, const float* v, const int64_t* offsets, int64_t n_events,
                 ho_cand_t* cands, int32_t* n_found, int32_t* labels, uint64_t* digest, int32_t* acc_out)
{
    const size_t nb = (size_t)p->n_theta * p->n_rho;
    const int K = p->max_candidates;
    int32_t* acc = (int32_t*)malloc(sizeof(int32_t) * nb);
    ho_cand_t* tmp = (ho_cand_t*)malloc(sizeof(ho_cand_t) * (size_t)K);
    int rc = HO_OK;
    if (!acc || !tmp) { free(acc); free(tmp); return HO_ENOMEM; }
    for (int64_t e = 0; e < n_events; ++e) {
        const int64_t a = offsets[e], n = offsets[e + 1] - offsets[e];
        int r = ho_vote_event(p, u + a, v + a, n, acc);
        if (r != HO_OK && rc == HO_OK) rc = r;
        if (digest) digest[e] = ho_digest(acc, p->n_theta, p->n_rho);
        if (acc_out) memcpy(acc_out + (size_t)e * nb, acc, sizeof(int32_t) * nb);
        if (cands || labels) {
            int32_t nf = 0;
            ho_cand_t* out = cands ? cands + (size_t)e * K : tmp;
            r = ho_find_clusters_event(p, acc, out, &nf);
            if (r != HO_OK && rc == HO_OK) rc = r;
            if (n_found) n_found[e] = nf;
            if (labels) {
                r = ho_assign_event(p, u + a, v + a, n, out, nf < K ? nf : K, labels + a);
                if (r != HO_OK && rc == HO_OK) rc = r;
            }
        }
    }
    free(acc); free(tmp);
    return rc;
}
