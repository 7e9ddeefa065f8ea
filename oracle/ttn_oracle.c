/*
 * ttn_oracle.c -- CPU ORACLE for the tropical tensor-network sweep.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2008_06888_b200/csrc/ and neither includes the other.
 *
 * What it computes (all citations are /root/reference/PAPER.md line numbers):
 *
 *   E(sigma) = - sum_{<ij>} J_ij sigma_i sigma_j - sum_i h_i sigma_i      Eq. (1)
 *   E0 = min_sigma E(sigma),  g = #{sigma : E(sigma) = E0},  one sigma* in argmin
 *   ("exact", abstract PAPER.md:23).  The tropical contraction returns max(-E) = -E0
 *    and the counting tuple of Eq. (4) PAPER.md:78-83 returns g.
 *
 * Two independent realisations:
 *
 *   O-brute  ttn_oracle_brute_ising / ttn_oracle_brute_potts3
 *            the definition written out: enumerate every configuration, evaluate
 *            Eq. (1) (or the Potts energy) term by term in double, keep the minimum,
 *            the number of exact ties and the lowest-index minimiser.
 *
 *   O-dp     ttn_oracle_dp_ising / ttn_oracle_dp_potts3
 *            site-by-site ("broken line") transfer dynamic programming in the
 *            (max,+) semiring of Eq. (2) PAPER.md:57 with the counting tuple of
 *            Eq. (4) PAPER.md:80.  The frontier holds the q^L joint states of the L
 *            most recently placed spins; placing site (r,c) contracts the bond to
 *            (r-1,c) (tensor (A2)), the bond to (r,c-1) (diagonal gate
 *            (A4)) and the field (A3).  It is a legal
 *            order of the same contraction because diagonal gates commute
 *            ("The order of operation of these diagonal gates ... can be arbitrary",
 *            PAPER.md:118); it is deliberately NOT the gate-then-diagonal row order
 *            of the CUDA path.  Energies are double (exact for integer couplings),
 *            counts are unsigned 128-bit with checked addition (status 2 on
 *            overflow).  Ties: exact == on double (Eq. (4) "if x1 = x2").
 *            Configuration: every site step records, per new frontier state, which
 *            old digit won the (+) (the first argument on ties, footnote [49]
 *            PAPER.md:201); the end picks the lowest-index maximiser and walks the
 *            records back ("caching intermediate contraction results and
 *            backtracking").
 *
 * Conventions: L x L lattice, open boundaries,
 * site (r,c); Jh[r*(L-1)+c] couples (r,c)-(r,c+1); Jv[r*L+c] couples (r,c)-(r+1,c);
 * h[r*L+c]; Ising index bit 0 <-> sigma=+1, bit 1 <-> sigma=-1 ((A3): first index
 * carries +h).  Potts (App. C, in BASELINE.json's reading
 * E = -sum J delta(s_i,s_j)): colour t in {0,1,2}, no fields.
 *
 * Pins (tests/test_oracle_*.py): O-dp == O-brute on all small sizes; ferromagnet
 * closed form; free spins; decoupled chains; gauge / transpose / reflection
 * invariance; proper 3-colouring counts of grid graphs; finite-difference in h.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libttn_oracle.so ttn_oracle.c
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef unsigned __int128 u128;

#define ORACLE_OK 0
#define ORACLE_EINVAL 1
#define ORACLE_EOVERFLOW 2
#define ORACLE_ENOMEM 3

static inline double spin_of_bit(unsigned b) { return b ? -1.0 : 1.0; } /* (A3) PAPER.md:247 */

/* ------------------------------------------------------------------------------------------
 * O-brute, Ising.  Configuration index k in [0, 2^(L*L)): bit (r*L+c) of k is the index bit
 * of site (r,c).  Requires L*L <= 30.
 * ---------------------------------------------------------------------------------------- */
static double ising_energy_of(int L, const double *Jh, const double *Jv, const double *h,
                              uint64_t k) {
    /* Eq. (1), term by term. */
    double E = 0.0;
    for (int r = 0; r < L; ++r)
        for (int c = 0; c < L; ++c) {
            double s = spin_of_bit((unsigned)((k >> (r * L + c)) & 1u));
            if (c + 1 < L) {
                double t = spin_of_bit((unsigned)((k >> (r * L + c + 1)) & 1u));
                E -= Jh[r * (L - 1) + c] * s * t;
            }
            if (r + 1 < L) {
                double t = spin_of_bit((unsigned)((k >> ((r + 1) * L + c)) & 1u));
                E -= Jv[r * L + c] * s * t;
            }
            if (h) E -= h[r * L + c] * s;
        }
    return E;
}

/* Evaluate Eq. (1) for a given +-1 configuration (used by tests to score returned sigma). */
double ttn_oracle_ising_energy(int L, const double *Jh, const double *Jv, const double *h,
                               const int8_t *sigma) {
    double E = 0.0;
    for (int r = 0; r < L; ++r)
        for (int c = 0; c < L; ++c) {
            double s = (double)sigma[r * L + c];
            if (c + 1 < L) E -= Jh[r * (L - 1) + c] * s * (double)sigma[r * L + c + 1];
            if (r + 1 < L) E -= Jv[r * L + c] * s * (double)sigma[(r + 1) * L + c];
            if (h) E -= h[r * L + c] * s;
        }
    return E;
}

int ttn_oracle_brute_ising(int L, const double *Jh, const double *Jv, const double *h,
                           double *E0, uint64_t *g, int8_t *sigma) {
    if (L < 1 || L * L > 30 || !Jh || !Jv || !E0 || !g) return ORACLE_EINVAL;
    const uint64_t ncfg = 1ull << (L * L);
    double best = INFINITY;
    uint64_t cnt = 0, arg = 0;
#pragma omp parallel
    {
        double lbest = INFINITY;
        uint64_t lcnt = 0, larg = 0;
#pragma omp for schedule(static)
        for (uint64_t k = 0; k < ncfg; ++k) {
            double E = ising_energy_of(L, Jh, Jv, h, k);
            if (E < lbest) { lbest = E; lcnt = 1; larg = k; }
            else if (E == lbest) { lcnt += 1; }
        }
#pragma omp critical
        {
            if (lbest < best) { best = lbest; cnt = lcnt; arg = larg; }
            else if (lbest == best) { cnt += lcnt; if (lcnt && larg < arg) arg = larg; }
        }
    }
    *E0 = best;
    *g = cnt;
    if (sigma)
        for (int i = 0; i < L * L; ++i) sigma[i] = ((arg >> i) & 1u) ? -1 : 1;
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * O-brute, 3-state Potts, E = - sum_<ij> J_ij delta(t_i, t_j).  Requires L*L <= 18.
 * ---------------------------------------------------------------------------------------- */
int ttn_oracle_brute_potts3(int L, const double *Jh, const double *Jv, double *E0, uint64_t *g,
                            int8_t *colour) {
    if (L < 1 || L * L > 18 || !Jh || !Jv || !E0 || !g) return ORACLE_EINVAL;
    const int N = L * L;
    uint64_t ncfg = 1;
    for (int i = 0; i < N; ++i) ncfg *= 3;
    double best = INFINITY;
    uint64_t cnt = 0, arg = 0;
#pragma omp parallel
    {
        double lbest = INFINITY;
        uint64_t lcnt = 0, larg = 0;
        int8_t t[32];
#pragma omp for schedule(static)
        for (uint64_t k = 0; k < ncfg; ++k) {
            uint64_t kk = k;
            for (int i = 0; i < N; ++i) { t[i] = (int8_t)(kk % 3); kk /= 3; }
            double E = 0.0;
            for (int r = 0; r < L; ++r)
                for (int c = 0; c < L; ++c) {
                    if (c + 1 < L && t[r * L + c] == t[r * L + c + 1]) E -= Jh[r * (L - 1) + c];
                    if (r + 1 < L && t[r * L + c] == t[(r + 1) * L + c]) E -= Jv[r * L + c];
                }
            if (E < lbest) { lbest = E; lcnt = 1; larg = k; }
            else if (E == lbest) { lcnt += 1; }
        }
#pragma omp critical
        {
            if (lbest < best) { best = lbest; cnt = lcnt; arg = larg; }
            else if (lbest == best) { cnt += lcnt; if (lcnt && larg < arg) arg = larg; }
        }
    }
    *E0 = best;
    *g = cnt;
    if (colour)
        for (int i = 0; i < N; ++i) { colour[i] = (int8_t)(arg % 3); arg /= 3; }
    return ORACLE_OK;
}

double ttn_oracle_potts3_energy(int L, const double *Jh, const double *Jv, const int8_t *colour) {
    double E = 0.0;
    for (int r = 0; r < L; ++r)
        for (int c = 0; c < L; ++c) {
            if (c + 1 < L && colour[r * L + c] == colour[r * L + c + 1]) E -= Jh[r * (L - 1) + c];
            if (r + 1 < L && colour[r * L + c] == colour[(r + 1) * L + c]) E -= Jv[r * L + c];
        }
    return E;
}

/* ------------------------------------------------------------------------------------------
 * O-dp, Ising.  F[s], s in [0,2^L): tropical number x (= max of -E over everything already
 * summed out) and, if want_count, the counting-tuple n of Eq. (4).
 *   want_count = 0: energy only (8 bytes per state; L = 32 needs 34 GB)
 *   want_config != 0: also records L*L * 2^L decision bits and fills sigma[L*L] (+1/-1)
 * g is returned as two 64-bit halves.
 * ---------------------------------------------------------------------------------------- */
int ttn_oracle_dp_ising(int L, const double *Jh, const double *Jv, const double *h,
                        int want_count, int want_config, double *E0, uint64_t *g_lo,
                        uint64_t *g_hi, int8_t *sigma) {
    if (L < 1 || L > 40 || !Jh || !Jv || !E0) return ORACLE_EINVAL;
    if (want_count && (!g_lo || !g_hi)) return ORACLE_EINVAL;
    if (want_config && !sigma) return ORACLE_EINVAL;
    const uint64_t NS = 1ull << L;
    double *X = (double *)malloc(NS * sizeof(double));
    u128 *Nn = want_count ? (u128 *)malloc(NS * sizeof(u128)) : NULL;
    /* choice[(r*L+c)*NS + s'] = old digit b that won at new state s' (bit-packed) */
    uint8_t *choice = NULL;
    const uint64_t words_per_site = (NS + 7) / 8;
    if (want_config) choice = (uint8_t *)calloc((size_t)L * L * words_per_site, 1);
    if (!X || (want_count && !Nn) || (want_config && !choice)) {
        free(X); free(Nn); free(choice);
        return ORACLE_ENOMEM;
    }
    int overflow = 0;

    /* initial state: the tropical one, (0,0)^{(x)L}; counting one = (0,1). The
       frontier starts with zero placed spins (a single entry) and grows during row 0. */
    X[0] = 0.0;
    if (Nn) Nn[0] = 1;

    /* ---- row 0: frontier grows from 2^c to 2^(c+1) entries --------------------------------- */
    for (int c = 0; c < L; ++c) {
        const uint64_t half = 1ull << c;
        const double hh = h ? h[0 * L + c] : 0.0;
        const double jl = (c > 0) ? Jh[0 * (L - 1) + (c - 1)] : 0.0;
        /* new digit c = 1 first (reads X[s], writes X[s+half]); then digit c = 0 in place */
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < half; ++s) {
            double left = (c > 0) ? spin_of_bit((unsigned)((s >> (c - 1)) & 1u)) : 0.0;
            double w0 = jl * left * (+1.0) + hh * (+1.0);
            double w1 = jl * left * (-1.0) + hh * (-1.0);
            double x = X[s];
            X[s + half] = x + w1;   /* (.) of Eq. (2): x (.) w = x + w */
            X[s] = x + w0;
            if (Nn) Nn[s + half] = Nn[s]; /* n * 1, Eq. (4) */
        }
    }

    /* ---- rows 1..L-1: replace digit c ------------------------------------------------------ */
    for (int r = 1; r < L; ++r)
        for (int c = 0; c < L; ++c) {
            const uint64_t bit = 1ull << c;
            const double jv = Jv[(r - 1) * L + c];
            const double jl = (c > 0) ? Jh[r * (L - 1) + (c - 1)] : 0.0;
            const double hh = h ? h[r * L + c] : 0.0;
            uint8_t *ch = choice ? choice + (size_t)(r * L + c) * words_per_site : NULL;
#pragma omp parallel for schedule(static) reduction(| : overflow)
            for (uint64_t p = 0; p < NS / 2; ++p) {
                /* s0: pair index p with a 0 inserted at bit c */
                uint64_t s0 = ((p >> c) << (c + 1)) | (p & (bit - 1));
                uint64_t s1 = s0 | bit;
                double left = (c > 0) ? spin_of_bit((unsigned)((s0 >> (c - 1)) & 1u)) : 0.0;
                double xo[2] = { X[s0], X[s1] };
                u128 no[2] = { Nn ? Nn[s0] : 0, Nn ? Nn[s1] : 0 };
                for (unsigned bn = 0; bn < 2; ++bn) {          /* new digit b' */
                    double sn = spin_of_bit(bn);
                    double diag = jl * left * sn + hh * sn;   /* (A4) + (A3) */
                    /* (+) over old digit b of F[b] (.) (A2)[b][b'] */
                    double cand0 = xo[0] + jv * spin_of_bit(0) * sn;
                    double cand1 = xo[1] + jv * spin_of_bit(1) * sn;
                    double xm; u128 nm; unsigned win;
                    if (cand0 > cand1)      { xm = cand0; nm = no[0]; win = 0; }
                    else if (cand0 < cand1) { xm = cand1; nm = no[1]; win = 1; }
                    else {                                  /* exact tie, Eq. (4) */
                        xm = cand0; win = 0;                 /* first argument, [49] */
                        nm = no[0] + no[1];
                        if (Nn && nm < no[0]) overflow |= 1;
                    }
                    uint64_t sd = bn ? s1 : s0;
                    X[sd] = xm + diag;
                    if (Nn) Nn[sd] = nm;
                    if (ch && win) {
                        /* two threads may share a byte only if their sd differ by < 8 and
                           belong to different p; use an atomic or */
#pragma omp atomic
                        ch[sd >> 3] |= (uint8_t)(1u << (sd & 7));
                    }
                }
            }
        }

    /* ---- final (+) over the frontier: contraction with the end state (0,0)^L, PAPER.md:105 -- */
    double xm = -INFINITY; u128 nm = 0; uint64_t arg = 0;
    for (uint64_t s = 0; s < NS; ++s) {
        if (X[s] > xm) { xm = X[s]; nm = Nn ? Nn[s] : 0; arg = s; }
        else if (X[s] == xm && Nn) { u128 t = nm + Nn[s]; if (t < nm) overflow |= 1; nm = t; }
    }
    *E0 = (xm == 0.0) ? 0.0 : -xm;
    if (want_count) { *g_lo = (uint64_t)nm; *g_hi = (uint64_t)(nm >> 64); }

    if (want_config) {
        uint64_t s = arg;
        for (int r = L - 1; r >= 1; --r)
            for (int c = L - 1; c >= 0; --c) {
                const uint8_t *ch = choice + (size_t)(r * L + c) * words_per_site;
                sigma[r * L + c] = ((s >> c) & 1u) ? -1 : 1;
                unsigned b = (ch[s >> 3] >> (s & 7)) & 1u;
                s = (s & ~(1ull << c)) | ((uint64_t)b << c);
            }
        for (int c = 0; c < L; ++c) sigma[c] = ((s >> c) & 1u) ? -1 : 1;
    }
    free(X); free(Nn); free(choice);
    return overflow ? ORACLE_EOVERFLOW : ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------
 * O-dp, 3-state Potts (App. C; E = -sum J delta).  Frontier index in base 3.
 * ---------------------------------------------------------------------------------------- */
int ttn_oracle_dp_potts3(int L, const double *Jh, const double *Jv, int want_count,
                         int want_config, double *E0, uint64_t *g_lo, uint64_t *g_hi,
                         int8_t *colour) {
    if (L < 1 || L > 24 || !Jh || !Jv || !E0) return ORACLE_EINVAL;
    if (want_count && (!g_lo || !g_hi)) return ORACLE_EINVAL;
    if (want_config && !colour) return ORACLE_EINVAL;
    uint64_t pw[32];
    pw[0] = 1;
    for (int i = 1; i <= L; ++i) pw[i] = pw[i - 1] * 3;
    const uint64_t NS = pw[L];
    double *X = (double *)malloc(NS * sizeof(double));
    u128 *Nn = want_count ? (u128 *)malloc(NS * sizeof(u128)) : NULL;
    uint8_t *choice = NULL; /* one byte per (site, new state): winning old colour */
    if (want_config) choice = (uint8_t *)calloc((size_t)L * L * NS, 1);
    if (!X || (want_count && !Nn) || (want_config && !choice)) {
        free(X); free(Nn); free(choice);
        return ORACLE_ENOMEM;
    }
    int overflow = 0;
    X[0] = 0.0;
    if (Nn) Nn[0] = 1;

    for (int c = 0; c < L; ++c) { /* row 0: grow */
        const uint64_t sz = pw[c];
        const double jl = (c > 0) ? Jh[c - 1] : 0.0;
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < sz; ++s) {
            int left = (c > 0) ? (int)((s / pw[c - 1]) % 3) : -1;
            double x = X[s];
            u128 n = Nn ? Nn[s] : 0;
            for (int t = 2; t >= 0; --t) { /* t = 0 last: it overwrites X[s] */
                X[s + (uint64_t)t * sz] = x + ((left == t) ? jl : 0.0);
                if (Nn) Nn[s + (uint64_t)t * sz] = n;
            }
        }
    }

    for (int r = 1; r < L; ++r)
        for (int c = 0; c < L; ++c) {
            const uint64_t st = pw[c];
            const double jv = Jv[(r - 1) * L + c];
            const double jl = (c > 0) ? Jh[r * (L - 1) + (c - 1)] : 0.0;
            uint8_t *ch = choice ? choice + (size_t)(r * L + c) * NS : NULL;
#pragma omp parallel for schedule(static) reduction(| : overflow)
            for (uint64_t p = 0; p < NS / 3; ++p) {
                uint64_t lo = p % st, hi = p / st;
                uint64_t s0 = hi * st * 3 + lo;
                int left = (c > 0) ? (int)((lo / pw[c - 1]) % 3) : -1;
                double xo[3]; u128 no[3];
                for (int t = 0; t < 3; ++t) { xo[t] = X[s0 + t * st]; no[t] = Nn ? Nn[s0 + t * st] : 0; }
                for (int tn = 0; tn < 3; ++tn) {
                    double xm = -INFINITY; u128 nm = 0; int win = 0;
                    for (int t = 0; t < 3; ++t) {
                        double cand = xo[t] + ((t == tn) ? jv : 0.0); /* 3x3 gate, App. C */
                        if (cand > xm) { xm = cand; nm = no[t]; win = t; }
                        else if (cand == xm) { u128 q = nm + no[t]; if (Nn && q < nm) overflow |= 1; nm = q; }
                    }
                    X[s0 + tn * st] = xm + ((left == tn) ? jl : 0.0);
                    if (Nn) Nn[s0 + tn * st] = nm;
                    if (ch) ch[s0 + tn * st] = (uint8_t)win;
                }
            }
        }

    double xm = -INFINITY; u128 nm = 0; uint64_t arg = 0;
    for (uint64_t s = 0; s < NS; ++s) {
        if (X[s] > xm) { xm = X[s]; nm = Nn ? Nn[s] : 0; arg = s; }
        else if (X[s] == xm && Nn) { u128 t = nm + Nn[s]; if (t < nm) overflow |= 1; nm = t; }
    }
    *E0 = (xm == 0.0) ? 0.0 : -xm;
    if (want_count) { *g_lo = (uint64_t)nm; *g_hi = (uint64_t)(nm >> 64); }

    if (want_config) {
        uint64_t s = arg;
        for (int r = L - 1; r >= 1; --r)
            for (int c = L - 1; c >= 0; --c) {
                const uint8_t *ch = choice + (size_t)(r * L + c) * NS;
                int t = (int)((s / pw[c]) % 3);
                colour[r * L + c] = (int8_t)t;
                int b = ch[s];
                s = s - (uint64_t)t * pw[c] + (uint64_t)b * pw[c];
            }
        for (int c = 0; c < L; ++c) colour[c] = (int8_t)((s / pw[c]) % 3);
    }
    free(X); free(Nn); free(choice);
    return overflow ? ORACLE_EOVERFLOW : ORACLE_OK;
}

int ttn_oracle_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
    n = omp_get_max_threads();
#endif
    return n;
}
