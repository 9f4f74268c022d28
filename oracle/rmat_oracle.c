/*
 * oracle/rmat_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU evaluation of the R-matrix of
 * PSTGF (arxiv 1909.07321), eq. 4, PAPER.md:108:
 *
 *     R_nm(E) = 1/(2 r0) * sum_{k=1..M} w_nk w_mk / (E_k - E)
 *
 * with r0 == a the R-matrix radius (record RA), w_nk the
 * surface amplitudes (record WMAT; n over channels, k over the
 * Hamiltonian size) and E_k the R-matrix poles (record
 * VALUE).
 *
 * The method reaches exactly this result (up to rounding order), so the
 * oracle is the definition written out: every one of the n_chan^2 entries of
 * every energy is an independent k-ascending sum in FP64, each term
 * (w_nk*w_mk)/(E_k-E), added with Neumaier's compensated summation
 * (north_star: "plain, slow CPU triple loop in FP64 with compensated (Kahan)
 * summation").  No blocking, no symmetry shortcut, no reordering.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code with
 * paper_1909_07321_b200/csrc and neither side includes the other.
 *
 * Pins (tests/test_oracle_pins.py): exact rational brute force, the hand
 * example of tests/golden/eq4_hand_example.txt, the single-pole closed form,
 * symmetry, definiteness, the resolvent identity, exact scalings, block
 * structure, additivity, degenerate poles vs. a library SYRK; the leading
 * dimension (ldw > n_poles) and the diagonal addend have pins of their own.
 * Nothing in this file is "parity unpinned".
 *
 * The optional diagonal addend (diag_add[e][n], added to R_nn after the
 * division by 2a) is where a caller puts a Buttle correction: PAPER.md lists
 * that correction's data (records NBUTD/EBUTD/CBUTD, PAPER.md:524-528, :544,
 * file DBUT :581-583) but not its formula, so the oracle -- like the library
 * -- takes the diagonal from the caller and only defines where it goes.
 *
 * Build: gcc -O2 -std=c11 -fno-fast-math -ffp-contract=off -fopenmp -fPIC -shared
 * (-ffp-contract=off keeps the compensation from being fused away).
 */
#include <math.h>
#include <stddef.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* One entry of eq. 4 at one energy: k ascending, Neumaier-compensated. */
static double eq4_entry(const double *w_n, const double *w_m, const double *E_k,
                        int n_poles, double E, double a)
{
    double s = 0.0, c = 0.0;
    for (int k = 0; k < n_poles; ++k) {
        double t = (w_n[k] * w_m[k]) / (E_k[k] - E);
        double u = s + t;
        if (fabs(s) >= fabs(t))
            c += (s - u) + t;
        else
            c += (t - u) + s;
        s = u;
    }
    return (s + c) / (2.0 * a);
}

/*
 * R_out[e][n][m] for e in [0,n_E), n,m in [0,n_chan): dense, row-major.
 * W is row-major [n_chan][ldw] with k contiguous (reading R6).
 * diag_add (may be NULL) is [n_E][n_chan]: R_out[e][n][n] += diag_add[e][n],
 * one rounded addition after the division by 2a.
 * threads <= 1 runs serially; threads > 1 splits the energy loop only
 * (the arithmetic of each entry is unchanged).  Returns 0, or 1 on bad
 * arguments.
 */
int oracle_rmat_form(const double *W, long long ldw, const double *E_k,
                     const double *energies, int n_chan, int n_poles, int n_E,
                     double a, const double *diag_add, double *R_out, int threads)
{
    if (n_chan < 0 || n_poles < 0 || n_E < 0 || ldw < n_poles) return 1;
    if (n_chan == 0 || n_E == 0) return 0;
    if (!W && n_poles > 0) return 1;
    if (!energies || !R_out) return 1;
    (void)threads;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 1 ? threads : 1)
#endif
    for (int e = 0; e < n_E; ++e) {
        double E = energies[e];
        double *R = R_out + (size_t)e * (size_t)n_chan * (size_t)n_chan;
        for (int n = 0; n < n_chan; ++n)
            for (int m = 0; m < n_chan; ++m)
                R[(size_t)n * n_chan + m] =
                    eq4_entry(W + (size_t)n * ldw, W + (size_t)m * ldw, E_k, n_poles, E, a);
        if (diag_add)
            for (int n = 0; n < n_chan; ++n)
                R[(size_t)n * n_chan + n] += diag_add[(size_t)e * n_chan + n];
    }
    return 0;
}

/*
 * The same entries, one at a time: out[s] = R[e_idx[s]][n_idx[s]][m_idx[s]] of eq. 4
 * for s in [0,n_samples).  For waves too large to evaluate densely
 * (the paper's 7261 x 106 661 case: one dense energy is 2.8e12 terms)
 * the parity tests check sampled outputs this way.  Same eq4_entry as above, so every
 * pin of oracle_rmat_form pins this too (tests check the two agree bitwise).
 * Returns 0, 1 on bad arguments, 2 on an index out of range.
 */
int oracle_rmat_entries(const double *W, long long ldw, const double *E_k,
                        const double *energies, int n_chan, int n_poles, int n_E,
                        double a, long long n_samples, const int *e_idx, const int *n_idx,
                        const int *m_idx, double *out, int threads)
{
    if (n_chan < 0 || n_poles < 0 || n_E < 0 || ldw < n_poles || n_samples < 0) return 1;
    if (n_samples == 0) return 0;
    if ((!W && n_poles > 0) || !energies || !e_idx || !n_idx || !m_idx || !out) return 1;
    for (long long s = 0; s < n_samples; ++s)
        if (e_idx[s] < 0 || e_idx[s] >= n_E || n_idx[s] < 0 || n_idx[s] >= n_chan ||
            m_idx[s] < 0 || m_idx[s] >= n_chan)
            return 2;
    (void)threads;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16) num_threads(threads > 1 ? threads : 1)
#endif
    for (long long s = 0; s < n_samples; ++s)
        out[s] = eq4_entry(W + (size_t)n_idx[s] * ldw, W + (size_t)m_idx[s] * ldw, E_k, n_poles,
                           energies[e_idx[s]], a);
    return 0;
}

/* Threads the OpenMP runtime would use by default (for reporting "cores"). */
int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
