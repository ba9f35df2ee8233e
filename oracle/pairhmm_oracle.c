/*
 * ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, literal CPU PairHMM forward (three matrices M, I, D), written from the equations of
 * arxiv/paper_2606_25738 ("Endeavor"), reference/PAPER.md:
 *   Eq.1  initialisation,
 *   Eq.2  recurrence,
 *   Eq.3  emission prior P(r_i|h_j),
 *   Eq.4  likelihood L = sum_j M_{l,j} + I_{l,j}.
 * It is deliberately NOT the paper's row-wise reformulation (Eq.6-7): the CUDA path implements that
 * reformulation, so parity against this file also checks the re-derivation.  No blocking, fusion or
 * reordering: rows i = 1..l, columns j = 1..k, three rolling rows.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call
 * this.  It shares no code with paper_2606_25738_b200/csrc.
 *
 * Arithmetic: IEEE double.  To never underflow, after every completed row the three rows are
 * multiplied by an exact power of two 2^-e (e = ilogb of the row maximum) and e is added to a
 * separate integer exponent; the result is log10(sum) + E*log10(2) - log10(C).   (The paper instead
 * relies on the large constant C = 2^1020, Eq.1; rescale=0 reproduces that behaviour.)
 *
 * Readings of the paper used here:
 *   G1  D_{0,j} = C/k for j = 0..k (row-0 rule wins at (0,0): PAPER.md:241 gives
 *       M_{1,j} = p_{1,j} T_DM C/k for every j); M, I, D are 0 in column 0 for i >= 1.
 *   G4  mismatch prior is exactly eps/3 (Eq.3), not 0.33 (Listing 2).
 *   G5  qualities are raw Phred values: eps = 10^(-Q/10) (Eq.3's "-33" is the FASTQ offset).
 *   G6  T_MM_i = 1 - iota_i - d_i, T_MI_i = iota_i, T_MD_i = d_i with iota_i = 10^(-Qi_i/10),
 *       d_i = 10^(-Qd_i/10) of read position i.
 *   G7  T_II_i = T_DD_i = gamma_i = 10^(-Qg_i/10), T_IM_i = T_DM_i = 1 - gamma_i, taken at the row
 *       of the cell being written (gamma = 0.1 at GCP 10, the paper's constants).
 *       Non-uniform GCP is NOT pinned by the paper ("parity unpinned" for that case only).
 *   G8  the sum of Eq.4 runs over j = 1..k.
 *   G17 P(r_i|h_j) compares bytes literally.  n_wildcard != 0 (off in every BASELINE.json config; the GATK-style
 *       compatibility switch of SURVEY.md section 8(f) item 3): an 'N' in either sequence matches anything.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force path enumeration, closed forms
 * (1-base read, 1-base haplotype, gapless limit), the paper's first-row formula,
 * Eq.6 identity on stored rows, bounds, invariants, golden fixtures, a log-space second
 * implementation.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_E_ARG -1
#define ORACLE_E_NOMEM -2

/* One pair.  log2C: the scale constant is C = 2^log2C (Eq.1 uses 1020; 0 gives C = 1).
 * rescale != 0: per-row power-of-two rescaling with a separate exponent.
 * dump (optional, may be NULL): 3*(l+1)*(k+1) doubles, the matrices M, I, D (in that order, row
 * major, row 0 and column 0 included) holding mantissas; dump_exp (l+1 ints) the power-of-two
 * exponent of each row, so that true value = dump * 2^dump_exp[i] (all 0 when rescale == 0). */
static int n_wildcard_flag = 0; /* set through phmm_oracle_set_n_wildcard; read-only while a batch runs */
void phmm_oracle_set_n_wildcard(int on) { n_wildcard_flag = on ? 1 : 0; }

int phmm_oracle_pair(const uint8_t* read, const uint8_t* qb, const uint8_t* qi, const uint8_t* qd,
                     const uint8_t* qg, int64_t l, const uint8_t* hap, int64_t k, double log2C, int rescale,
                     double* out_log10, double* dump, int32_t* dump_exp) {
    if (!read || !qb || !qi || !qd || !qg || !hap || !out_log10 || l <= 0 || k <= 0) return ORACLE_E_ARG;
    size_t w = (size_t)k + 1;
    double* buf = (double*)malloc(sizeof(double) * 6 * w);
    if (!buf) return ORACLE_E_NOMEM;
    double *Mp = buf, *Ip = buf + w, *Dp = buf + 2 * w, *Mc = buf + 3 * w, *Ic = buf + 4 * w, *Dc = buf + 5 * w;
    const double C = ldexp(1.0, (int)log2C);
    int64_t E = 0; /* accumulated power-of-two exponent: true row = stored row * 2^E */

    /* Eq.1: M_{0,j} = I_{0,j} = 0, D_{0,j} = C/k (j = 0..k, reading G1) */
    for (int64_t j = 0; j <= k; j++) { Mp[j] = 0.0; Ip[j] = 0.0; Dp[j] = C / (double)k; }
    if (dump) {
        size_t plane = (size_t)(l + 1) * w;
        for (int64_t j = 0; j <= k; j++) { dump[j] = Mp[j]; dump[plane + j] = Ip[j]; dump[2 * plane + j] = Dp[j]; }
        if (dump_exp) dump_exp[0] = 0;
    }

    for (int64_t i = 1; i <= l; i++) {
        /* per-row probabilities from the Phred bytes of read position i (Eq.3; readings G5-G7) */
        const double eps = pow(10.0, -(double)qb[i - 1] / 10.0);
        const double iota = pow(10.0, -(double)qi[i - 1] / 10.0);
        const double del = pow(10.0, -(double)qd[i - 1] / 10.0);
        const double gam = pow(10.0, -(double)qg[i - 1] / 10.0);
        const double p_match = 1.0 - eps, p_mis = eps / 3.0;
        const double T_MM = 1.0 - iota - del, T_MI = iota, T_MD = del;
        const double T_II = gam, T_DD = gam, T_IM = 1.0 - gam, T_DM = 1.0 - gam;
        const uint8_t r = read[i - 1];

        Mc[0] = 0.0; Ic[0] = 0.0; Dc[0] = 0.0; /* Eq.1: column 0 is zero for i >= 1 */
        for (int64_t j = 1; j <= k; j++) {
            const int same = (r == hap[j - 1]) || (n_wildcard_flag && (r == 'N' || hap[j - 1] == 'N'));
            const double p = same ? p_match : p_mis;                                   /* Eq.3 */
            Mc[j] = p * (T_MM * Mp[j - 1] + T_IM * Ip[j - 1] + T_DM * Dp[j - 1]);      /* Eq.2 */
            Ic[j] = T_MI * Mp[j] + T_II * Ip[j];                                        /* Eq.2 */
            Dc[j] = T_MD * Mc[j - 1] + T_DD * Dc[j - 1];                                /* Eq.2 */
        }
        if (rescale) {
            double m = 0.0;
            for (int64_t j = 0; j <= k; j++) {
                if (Mc[j] > m) m = Mc[j];
                if (Ic[j] > m) m = Ic[j];
                if (Dc[j] > m) m = Dc[j];
            }
            if (m > 0.0 && isfinite(m)) {
                int e = ilogb(m);
                if (e != 0) {
                    for (int64_t j = 0; j <= k; j++) {
                        Mc[j] = ldexp(Mc[j], -e); Ic[j] = ldexp(Ic[j], -e); Dc[j] = ldexp(Dc[j], -e);
                    }
                    E += e;
                }
            }
        }
        if (dump) {
            size_t plane = (size_t)(l + 1) * w, row = (size_t)i * w;
            for (int64_t j = 0; j <= k; j++) { dump[row + j] = Mc[j]; dump[plane + row + j] = Ic[j]; dump[2 * plane + row + j] = Dc[j]; }
            if (dump_exp) dump_exp[i] = (int32_t)E;
        }
        double* t;
        t = Mp; Mp = Mc; Mc = t;
        t = Ip; Ip = Ic; Ic = t;
        t = Dp; Dp = Dc; Dc = t;
    }
    /* Eq.4: L = sum_{j=1..k} (M_{l,j} + I_{l,j}) / C */
    double sum = 0.0;
    for (int64_t j = 1; j <= k; j++) sum += Mp[j] + Ip[j];
    *out_log10 = log10(sum) + ((double)E - log2C) * 0.30102999566398119521373889472449;
    free(buf);
    return ORACLE_OK;
}

/* A batch in the CSR layout of include/pairhmm_b200.h (all host pointers), OpenMP over pairs only. */
int phmm_oracle_batch(int64_t n_pairs, const int32_t* pair_read, const int32_t* pair_hap,
                      const int64_t* read_off, const int64_t* hap_off, const uint8_t* read_bases,
                      const uint8_t* qual_base, const uint8_t* qual_ins, const uint8_t* qual_del,
                      const uint8_t* qual_gcp, const uint8_t* hap_bases, double log2C, int rescale,
                      int n_threads, double* out_log10) {
    if (n_pairs < 0 || !out_log10) return ORACLE_E_ARG;
    int rc_all = ORACLE_OK;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t p = 0; p < n_pairs; p++) {
        int64_t r = pair_read[p], h = pair_hap[p];
        int64_t ro = read_off[r], l = read_off[r + 1] - ro, ho = hap_off[h], k = hap_off[h + 1] - ho;
        int rc = phmm_oracle_pair(read_bases + ro, qual_base + ro, qual_ins + ro, qual_del + ro, qual_gcp + ro, l,
                                  hap_bases + ho, k, log2C, rescale, out_log10 + p, NULL, NULL);
        if (rc != ORACLE_OK) {
            #pragma omp critical
            rc_all = rc;
        }
    }
    return rc_all;
}

int phmm_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
