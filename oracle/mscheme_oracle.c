/* ORACLE (test infrastructure, not product code).
 *
 * Plain C restatement of oracle/mscheme_ref.py (same steps, same loop order, same
 * notation) so that whole configs finish in seconds.  It is cross-checked against the
 * pure-Python version in tests/test_oracle_pins.py.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header or table generator with paper_1412_5989_b200/csrc; the coupling coefficients it
 * uses come from oracle/cg_exact.py (exact rationals), passed in as a flat table.
 *
 * What it computes: PAPER.md:55-61 (section 3.1) -- each requested m-scheme element is
 * the coupling-coefficient-weighted sum of the coupled-JT elements of the matching
 * block, reached by nested loops over coupled angular momentum and isospin values.
 * Formulas: DESIGN.md "Readings" Q1-Q7, restated in
 * oracle/mscheme_ref.py's header.
 *
 * Loop order (fixed): J, T, J12, T12, J12', T12' ascending; plain double accumulation.
 * OpenMP over requests only (each request is independent).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int n_orb;
    const int32_t *orb_n, *orb_l, *orb_twoj;
    int n_sps;
    const int32_t *sps_orb, *sps_twom, *sps_twotz;
    /* exact CG table from oracle/cg_exact.py:CGTable */
    int cg_dim1, cg_dim2;
    const int64_t *cg_off;
    const double *cg_val;
} oracle_basis;

static int iabs(int x) { return x < 0 ? -x : x; }

/* <j1 m1 j2 m2|J M> by table lookup; integer selection rules first (all doubled). */
static double cg(const oracle_basis *B, int tj1, int tm1, int tj2, int tm2, int tJ, int tM)
{
    if (tm1 + tm2 != tM) return 0.0;
    if (tJ < iabs(tj1 - tj2) || tJ > tj1 + tj2 || ((tj1 + tj2 + tJ) & 1)) return 0.0;
    if (iabs(tm1) > tj1 || iabs(tm2) > tj2 || iabs(tM) > tJ) return 0.0;
    if (((tj1 + tm1) & 1) || ((tj2 + tm2) & 1) || ((tJ + tM) & 1)) return 0.0;
    if (tj1 >= B->cg_dim1 || tj2 >= B->cg_dim2) return NAN;
    int64_t o = B->cg_off[(int64_t)tj1 * B->cg_dim2 + tj2];
    if (o < 0) return NAN; /* table does not cover this pair: poison the result */
    int iJ = (tJ - iabs(tj1 - tj2)) / 2;
    return B->cg_val[o + ((int64_t)iJ * (tj1 + 1) + (tm1 + tj1) / 2) * (tj2 + 1) + (tm2 + tj2) / 2];
}

/* stable sort of k (<=3) particles by (orbital, sps) ascending; returns permutation sign */
static int canonicalise(const oracle_basis *B, int k, int32_t *s)
{
    int inv = 0;
    for (int i = 0; i < k; i++)
        for (int j = i + 1; j < k; j++) {
            int oi = B->sps_orb[s[i]], oj = B->sps_orb[s[j]];
            if (oi > oj || (oi == oj && s[i] > s[j])) inv++;
        }
    for (int i = 1; i < k; i++) { /* insertion sort = stable */
        int32_t x = s[i];
        int j = i - 1;
        while (j >= 0 && (B->sps_orb[s[j]] > B->sps_orb[x] || (B->sps_orb[s[j]] == B->sps_orb[x] && s[j] > x))) {
            s[j + 1] = s[j];
            j--;
        }
        s[j + 1] = x;
    }
    return (inv & 1) ? -1 : 1;
}

/* ---- table lookups: states of a channel are sorted ascending, so binary search ---- */
static int64_t key2(int a, int b) { return ((int64_t)a << 20) | b; }
static int64_t key3(int a, int b, int c, int J12, int T12)
{
    return ((((((int64_t)a << 12) | b) << 12 | c) << 8 | J12) << 1) | T12;
}
static int find(const int64_t *keys, int lo, int hi, int64_t k)
{ /* first index in [lo,hi) with keys[i] >= k (hi if none) */
    while (lo < hi) {
        int mid = (lo + hi) / 2;
        if (keys[mid] < k) lo = mid + 1; else hi = mid;
    }
    return lo;
}
static int row_of(const int64_t *keys, int s0, int s1, int64_t k)
{
    int i = find(keys, s0, s1, k);
    return (i < s1 && keys[i] == k) ? i - s0 : -1;
}
static int chan_of(int n_chan, const int32_t *cJ, const int32_t *cT, const int32_t *cP, int J, int T, int par)
{
    for (int c = 0; c < n_chan; c++)
        if (cJ[c] == J && cT[c] == T && cP[c] == par) return c;
    return -1;
}
static int cmp64(const void *x, const void *y)
{
    int64_t a = *(const int64_t *)x, b = *(const int64_t *)y;
    return (a > b) - (a < b);
}

/* ------------------------------------------------------------------ 2-body */
int oracle_mscheme_2b(const oracle_basis *B, int n_chan, const int32_t *chan_J, const int32_t *chan_T,
                      const int32_t *chan_par, const int32_t *chan_dim, const int64_t *chan_off,
                      const int32_t *state_a, const int32_t *state_b, const double *values, int64_t n,
                      const int32_t *req, double *out, uint8_t *mask, int64_t *nterms, int64_t *bad_count,
                      int n_threads)
{
    int64_t n_states = 0;
    int *s0 = (int *)malloc(sizeof(int) * (n_chan + 1));
    for (int c = 0; c < n_chan; c++) { s0[c] = (int)n_states; n_states += chan_dim[c]; }
    s0[n_chan] = (int)n_states;
    int64_t *keys = (int64_t *)malloc(sizeof(int64_t) * (n_states + 1));
    int64_t *tuples = (int64_t *)malloc(sizeof(int64_t) * (n_states + 1));
    for (int64_t i = 0; i < n_states; i++) tuples[i] = keys[i] = key2(state_a[i], state_b[i]);
    qsort(tuples, n_states, sizeof(int64_t), cmp64);
    int maxJ = 0;
    for (int c = 0; c < n_chan; c++) if (chan_J[c] > maxJ) maxJ = chan_J[c];
    int64_t bad = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 1024) reduction(+ : bad)
    for (int64_t i = 0; i < n; i++) {
        out[i] = 0.0;
        if (mask) mask[i] = 0;
        if (nterms) nterms[i] = 0;
        int32_t bra[2] = {req[4 * i], req[4 * i + 1]}, ket[2] = {req[4 * i + 2], req[4 * i + 3]};
        int oob = 0;
        for (int k = 0; k < 2; k++) oob |= bra[k] < 0 || bra[k] >= B->n_sps || ket[k] < 0 || ket[k] >= B->n_sps;
        if (oob) { bad++; continue; }                                            /* step 1 */
        if (bra[0] == bra[1] || ket[0] == ket[1]) continue;                      /* S1 */
        int Mb = 0, Mk = 0, Tb = 0, Tk = 0, Pb = 0, Pk = 0;
        for (int k = 0; k < 2; k++) {
            Mb += B->sps_twom[bra[k]]; Mk += B->sps_twom[ket[k]];
            Tb += B->sps_twotz[bra[k]]; Tk += B->sps_twotz[ket[k]];
            Pb += B->orb_l[B->sps_orb[bra[k]]]; Pk += B->orb_l[B->sps_orb[ket[k]]];
        }
        if (Mb != Mk || Tb != Tk || ((Pb ^ Pk) & 1)) continue;                   /* S2 S3 S4 */
        int sign = canonicalise(B, 2, bra) * canonicalise(B, 2, ket);            /* step 3 */
        int a = B->sps_orb[bra[0]], b = B->sps_orb[bra[1]], c = B->sps_orb[ket[0]], d = B->sps_orb[ket[1]];
        if (row_of(tuples, 0, (int)n_states, key2(a, b)) < 0 || row_of(tuples, 0, (int)n_states, key2(c, d)) < 0)
            continue;                                                            /* S6 */
        int ja = B->orb_twoj[a], jb = B->orb_twoj[b], jc = B->orb_twoj[c], jd = B->orb_twoj[d];
        int ma = B->sps_twom[bra[0]], mb = B->sps_twom[bra[1]], mc = B->sps_twom[ket[0]], md = B->sps_twom[ket[1]];
        int ta = B->sps_twotz[bra[0]], tb = B->sps_twotz[bra[1]], tc = B->sps_twotz[ket[0]], td = B->sps_twotz[ket[1]];
        int par = Pb & 1;
        double total = 0.0;
        int64_t nt = 0;
        for (int J = 0; J <= maxJ; J++) {                                        /* step 4 */
            if (2 * J < iabs(Mb) || 2 * J < iabs(ja - jb) || 2 * J > ja + jb || 2 * J < iabs(jc - jd) || 2 * J > jc + jd)
                continue;
            for (int T = 0; T <= 1; T++) {
                if (2 * T < iabs(Tb)) continue;
                int ch = chan_of(n_chan, chan_J, chan_T, chan_par, J, T, par);
                if (ch < 0) continue;
                int r = row_of(keys, s0[ch], s0[ch + 1], key2(a, b));
                int q = row_of(keys, s0[ch], s0[ch + 1], key2(c, d));
                if (r < 0 || q < 0) continue;
                double Bc = cg(B, ja, ma, jb, mb, 2 * J, Mb) * cg(B, 1, ta, 1, tb, 2 * T, Tb);
                double Kc = cg(B, jc, mc, jd, md, 2 * J, Mb) * cg(B, 1, tc, 1, td, 2 * T, Tb);
                total += Bc * Kc * values[chan_off[ch] + (int64_t)r * chan_dim[ch] + q];
                nt++;
            }
        }
        if (nt == 0) continue;                                                   /* S7 */
        double norm = sqrt((a == b ? 2.0 : 1.0) * (c == d ? 2.0 : 1.0));
        out[i] = sign * norm * total;
        if (mask) mask[i] = 1;
        if (nterms) nterms[i] = nt;
    }
    if (bad_count) *bad_count = bad;
    free(s0); free(keys); free(tuples);
    return 0;
}

/* ------------------------------------------------------------------ 3-body */
int oracle_mscheme_3b(const oracle_basis *B, int e3max, int n_chan, const int32_t *chan_twoJ,
                      const int32_t *chan_twoT, const int32_t *chan_par, const int32_t *chan_dim,
                      const int64_t *chan_off, const int32_t *state_a, const int32_t *state_b,
                      const int32_t *state_c, const int32_t *state_J12, const int32_t *state_T12,
                      const double *values, int64_t n, const int32_t *req, double *out, uint8_t *mask,
                      int64_t *nterms, int64_t *bad_count, int n_threads)
{
    int64_t n_states = 0;
    int *s0 = (int *)malloc(sizeof(int) * (n_chan + 1));
    for (int c = 0; c < n_chan; c++) { s0[c] = (int)n_states; n_states += chan_dim[c]; }
    s0[n_chan] = (int)n_states;
    int64_t *keys = (int64_t *)malloc(sizeof(int64_t) * (n_states + 1));
    int64_t *tuples = (int64_t *)malloc(sizeof(int64_t) * (n_states + 1));
    for (int64_t i = 0; i < n_states; i++) {
        keys[i] = key3(state_a[i], state_b[i], state_c[i], state_J12[i], state_T12[i]);
        tuples[i] = key3(state_a[i], state_b[i], state_c[i], 0, 0);
    }
    qsort(tuples, n_states, sizeof(int64_t), cmp64);
    int max_twoJ = 0;
    for (int c = 0; c < n_chan; c++) if (chan_twoJ[c] > max_twoJ) max_twoJ = chan_twoJ[c];
    int64_t bad = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : bad)
    for (int64_t i = 0; i < n; i++) {
        out[i] = 0.0;
        if (mask) mask[i] = 0;
        if (nterms) nterms[i] = 0;
        int32_t bra[3], ket[3];
        int oob = 0;
        for (int k = 0; k < 3; k++) {
            bra[k] = req[6 * i + k]; ket[k] = req[6 * i + 3 + k];
            oob |= bra[k] < 0 || bra[k] >= B->n_sps || ket[k] < 0 || ket[k] >= B->n_sps;
        }
        if (oob) { bad++; continue; }                                            /* step 1 */
        if (bra[0] == bra[1] || bra[0] == bra[2] || bra[1] == bra[2]) continue;  /* S1 */
        if (ket[0] == ket[1] || ket[0] == ket[2] || ket[1] == ket[2]) continue;
        int Mb = 0, Mk = 0, Tb = 0, Tk = 0, Pb = 0, Pk = 0, Eb = 0, Ek = 0;
        for (int k = 0; k < 3; k++) {
            int ob = B->sps_orb[bra[k]], ok = B->sps_orb[ket[k]];
            Mb += B->sps_twom[bra[k]]; Mk += B->sps_twom[ket[k]];
            Tb += B->sps_twotz[bra[k]]; Tk += B->sps_twotz[ket[k]];
            Pb += B->orb_l[ob]; Pk += B->orb_l[ok];
            Eb += 2 * B->orb_n[ob] + B->orb_l[ob]; Ek += 2 * B->orb_n[ok] + B->orb_l[ok];
        }
        if (Mb != Mk || Tb != Tk || ((Pb ^ Pk) & 1)) continue;                   /* S2 S3 S4 */
        if (Eb > e3max || Ek > e3max) continue;                                  /* S5 */
        int sign = canonicalise(B, 3, bra) * canonicalise(B, 3, ket);            /* step 3 */
        int a = B->sps_orb[bra[0]], b = B->sps_orb[bra[1]], c = B->sps_orb[bra[2]];
        int d = B->sps_orb[ket[0]], e = B->sps_orb[ket[1]], f = B->sps_orb[ket[2]];
        if (row_of(tuples, 0, (int)n_states, key3(a, b, c, 0, 0)) < 0 ||
            row_of(tuples, 0, (int)n_states, key3(d, e, f, 0, 0)) < 0)
            continue;                                                            /* S6 */
        int ja = B->orb_twoj[a], jb = B->orb_twoj[b], jc = B->orb_twoj[c];
        int jd = B->orb_twoj[d], je = B->orb_twoj[e], jf = B->orb_twoj[f];
        int ma = B->sps_twom[bra[0]], mb = B->sps_twom[bra[1]], mc = B->sps_twom[bra[2]];
        int md = B->sps_twom[ket[0]], me = B->sps_twom[ket[1]], mf = B->sps_twom[ket[2]];
        int ta = B->sps_twotz[bra[0]], tb = B->sps_twotz[bra[1]], tc = B->sps_twotz[bra[2]];
        int td = B->sps_twotz[ket[0]], te = B->sps_twotz[ket[1]], tf = B->sps_twotz[ket[2]];
        int par = Pb & 1;
        double total = 0.0;
        int64_t nt = 0;
        for (int twoJ = 1; twoJ <= max_twoJ; twoJ += 2) {                        /* step 4 */
            if (twoJ < iabs(Mb)) continue;
            for (int twoT = 1; twoT <= 3; twoT += 2) {
                if (twoT < iabs(Tb)) continue;
                int ch = chan_of(n_chan, chan_twoJ, chan_twoT, chan_par, twoJ, twoT, par);
                if (ch < 0) continue;
                const double *V = values + chan_off[ch];
                int dim = chan_dim[ch];
                for (int J12 = iabs(ja - jb) / 2; J12 <= (ja + jb) / 2; J12++) {
                    if (2 * J12 < iabs(ma + mb) || twoJ < iabs(2 * J12 - jc) || twoJ > 2 * J12 + jc) continue;
                    for (int T12 = 0; T12 <= 1; T12++) {
                        if (2 * T12 < iabs(ta + tb) || twoT < iabs(2 * T12 - 1) || twoT > 2 * T12 + 1) continue;
                        int r = row_of(keys, s0[ch], s0[ch + 1], key3(a, b, c, J12, T12));
                        if (r < 0) continue;
                        double Bc = cg(B, ja, ma, jb, mb, 2 * J12, ma + mb) * cg(B, 2 * J12, ma + mb, jc, mc, twoJ, Mb) *
                                    cg(B, 1, ta, 1, tb, 2 * T12, ta + tb) * cg(B, 2 * T12, ta + tb, 1, tc, twoT, Tb);
                        for (int J12p = iabs(jd - je) / 2; J12p <= (jd + je) / 2; J12p++) {
                            if (2 * J12p < iabs(md + me) || twoJ < iabs(2 * J12p - jf) || twoJ > 2 * J12p + jf) continue;
                            for (int T12p = 0; T12p <= 1; T12p++) {
                                if (2 * T12p < iabs(td + te) || twoT < iabs(2 * T12p - 1) || twoT > 2 * T12p + 1) continue;
                                int q = row_of(keys, s0[ch], s0[ch + 1], key3(d, e, f, J12p, T12p));
                                if (q < 0) continue;
                                double Kc = cg(B, jd, md, je, me, 2 * J12p, md + me) *
                                            cg(B, 2 * J12p, md + me, jf, mf, twoJ, Mb) *
                                            cg(B, 1, td, 1, te, 2 * T12p, td + te) *
                                            cg(B, 2 * T12p, td + te, 1, tf, twoT, Tb);
                                total += Bc * Kc * V[(int64_t)r * dim + q];
                                nt++;
                            }
                        }
                    }
                }
            }
        }
        if (nt == 0) continue;                                                   /* S7 */
        out[i] = sign * total;
        if (mask) mask[i] = 1;
        if (nterms) nterms[i] = nt;
    }
    if (bad_count) *bad_count = bad;
    free(s0); free(keys); free(tuples);
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
