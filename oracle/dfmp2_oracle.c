/*
 * oracle/dfmp2_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, explicit-loop FP64 CPU definition of the fragment-projected DF-MP2 energy of one
 * SIE embedding cluster.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  It shares no code, header, table or helper with the CUDA
 * path under paper_2412_18553_b200/ and neither imports the other.
 *
 * What it computes, in the paper's order and notation (citations are /root/reference/PAPER.md lines):
 *
 *   O1  unpack   (P|mu nu) = (P|nu mu) from packed mu>=nu storage, idx = mu(mu+1)/2 + nu
 *   O2  H^P_{i nu}  = sum_mu C_{mu i} (P|mu nu)                        } DF form of the cluster
 *   O3  B^P_{ia}    = sum_nu H^P_{i nu} C_{nu a}                       } integral projection Eq. S49 (L526)
 *   O4  (ia|jb)     = V^{ij}_{ab} = sum_P B^P_{ia} B^P_{jb}
 *   O5  t_{ij}^{ab} = (ia|jb) / (e_i + e_j - e_a - e_b)                Eq. S15-S16 (L348-L351):
 *                     t = -(ia|jb)/D, D = e_a+e_b-e_i-e_j, i.e. the same number
 *   O6  G_{i'i}     = sum_j sum_ab t_{i'j}^{ab} ( 2 (ia|jb) - (ib|ja) )
 *                     closed-shell 2t-t combination, Eq. S17-S18/S22 (L355-L357, L390);
 *                     only the FIRST occupied index of the amplitude carries i' (Eq. S44;
 *                     Eq. S50); MP2 has no singles (L378)
 *   O7  E_frag      = sum_{i i'} P_frag[i][i'] G[i'][i]               P_frag = C^f_{ii'} = sum_f C_if C_i'f,
 *                                                                     Eq. S45 (L505) / S59 (L569)
 *
 * No blocking, fusion or reordering beyond that: the loops below are the definition.  The aux dot
 * of O4 uses 8 explicit partial sums (still a plain loop); the (a,b), j and trace accumulations are
 * carried in long double so the oracle's own rounding sits far below the GPU's.
 *
 * NEXT-1 additions at the end of this file: O8 gamma_ij and O9 gamma_ab, occupied and virtual blocks of the MP2 1-RDM
 * (Eq. S18, S17), pinned in tests/test_oracle_rdm_pins.py.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): hand-worked 2x1 and 1x1 cases
 * (tests/golden/handworked.txt), closed form o=v=1, P=I == textbook closed-shell MP2 from brute-force
 * four-index integrals, fragment additivity, invariances, scalings.  No function here is unpinned.
 *
 * Build: gcc -O3 -march=x86-64-v3 -fopenmp -shared -fPIC (oracle/build.py). No -ffast-math.
 */
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int sie_oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void sie_oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* O1: one packed symmetric matrix -> full nao x nao (row-major). */
void sie_oracle_unpack(int nao, const double* Lp, double* Lfull) {
    for (int mu = 0; mu < nao; ++mu)
        for (int nu = 0; nu <= mu; ++nu) {
            double x = Lp[(size_t)mu * (mu + 1) / 2 + nu];
            Lfull[(size_t)mu * nao + nu] = x;
            Lfull[(size_t)nu * nao + mu] = x;
        }
}

/* aux dot with 8 explicit partial sums */
static double dot8(const double* x, const double* y, int n) {
    double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int p = 0;
    for (; p + 8 <= n; p += 8)
        for (int u = 0; u < 8; ++u) s[u] += x[p + u] * y[p + u];
    for (int u = 0; p < n; ++p, ++u) s[u] += x[p] * y[p];
    return ((s[0] + s[1]) + (s[2] + s[3])) + ((s[4] + s[5]) + (s[6] + s[7]));
}

/*
 * O1-O3 for the aux rows [p0,p1) of the packed tensor.
 *   C_occ [nao][nocc], C_vir [nao][nvir] row-major; Lp_block [(p1-p0)][nao(nao+1)/2];
 *   B [nocc][nvir][naux] row-major (aux index contiguous): entries B[i][a][P], P in [p0,p1) are written.
 * Returns 0, or 1 on allocation failure.
 */
int sie_oracle_transform(int nao, int nocc, int nvir, int naux, int p0, int p1,
                         const double* C_occ, const double* C_vir, const double* Lp_block, double* B) {
    const size_t np = (size_t)nao * (nao + 1) / 2;
    int fail = 0;
#pragma omp parallel
    {
        double* Lfull = (double*)malloc(sizeof(double) * (size_t)nao * nao);
        double* H = (double*)malloc(sizeof(double) * (size_t)nocc * nao);
        if (!Lfull || !H) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (int P = p0; P < p1; ++P) {
                sie_oracle_unpack(nao, Lp_block + (size_t)(P - p0) * np, Lfull);          /* O1 */
                for (int i = 0; i < nocc; ++i)                                             /* O2 */
                    for (int nu = 0; nu < nao; ++nu) {
                        long double s = 0.0L;
                        for (int mu = 0; mu < nao; ++mu)
                            s += (long double)(C_occ[(size_t)mu * nocc + i] * Lfull[(size_t)mu * nao + nu]);
                        H[(size_t)i * nao + nu] = (double)s;
                    }
                for (int i = 0; i < nocc; ++i)                                             /* O3 */
                    for (int a = 0; a < nvir; ++a) {
                        long double s = 0.0L;
                        for (int nu = 0; nu < nao; ++nu)
                            s += (long double)(H[(size_t)i * nao + nu] * C_vir[(size_t)nu * nvir + a]);
                        B[((size_t)i * nvir + a) * naux + P] = (double)s;
                    }
            }
        }
        free(Lfull);
        free(H);
    }
    return fail;
}

/*
 * O4-O6 restricted to j in [j0,j1):  G[i'][i] = sum_{j0<=j<j1} sum_ab t_{i'j}^{ab} (2 V^{ij}_{ab} - V^{ij}_{ba}).
 *   B [nocc][nvir][naux], e_occ[nocc], e_vir[nvir]; G [nocc][nocc] row-major, OVERWRITTEN.
 * The full G is the call with (j0,j1) = (0,nocc); slices add.  Returns 0, or 1 on allocation failure.
 */
int sie_oracle_pair_G(int nocc, int nvir, int naux, const double* B, const double* e_occ,
                      const double* e_vir, int j0, int j1, double* G) {
    const size_t vv = (size_t)nvir * nvir;
    double* Vj = (double*)malloc(sizeof(double) * (size_t)nocc * vv);      /* V^{ij}[a][b] for all i at fixed j */
    long double* Gl = (long double*)calloc((size_t)nocc * nocc, sizeof(long double));
    if (!Vj || !Gl) { free(Vj); free(Gl); return 1; }
    int fail = 0;
    for (int j = j0; j < j1; ++j) {
        /* O4 */
#pragma omp parallel for collapse(2) schedule(static)
        for (int i = 0; i < nocc; ++i)
            for (int a = 0; a < nvir; ++a) {
                const double* bia = B + ((size_t)i * nvir + a) * naux;
                double* v = Vj + (size_t)i * vv + (size_t)a * nvir;
                for (int b = 0; b < nvir; ++b) v[b] = dot8(bia, B + ((size_t)j * nvir + b) * naux, naux);
            }
#pragma omp parallel
        {
            double* t = (double*)malloc(sizeof(double) * vv);
            if (!t) {
#pragma omp atomic write
                fail = 1;
            }
#pragma omp barrier
            if (!fail) {
#pragma omp for schedule(dynamic, 1)
                for (int ip = 0; ip < nocc; ++ip) {
                    const double* Vip = Vj + (size_t)ip * vv;
                    for (int a = 0; a < nvir; ++a)                                          /* O5 */
                        for (int b = 0; b < nvir; ++b)
                            t[(size_t)a * nvir + b] =
                                Vip[(size_t)a * nvir + b] / (e_occ[ip] + e_occ[j] - e_vir[a] - e_vir[b]);
                    for (int i = 0; i < nocc; ++i) {                                        /* O6 */
                        const double* Vi = Vj + (size_t)i * vv;
                        long double s = 0.0L;
                        for (int a = 0; a < nvir; ++a)
                            for (int b = 0; b < nvir; ++b)
                                s += (long double)t[(size_t)a * nvir + b] *
                                     (2.0L * (long double)Vi[(size_t)a * nvir + b] - (long double)Vi[(size_t)b * nvir + a]);
                        Gl[(size_t)ip * nocc + i] += s;
                    }
                }
            }
            free(t);
        }
        if (fail) break;
    }
    for (size_t k = 0; k < (size_t)nocc * nocc; ++k) G[k] = (double)Gl[k];
    free(Vj);
    free(Gl);
    return fail;
}

/* O7: E_frag = sum_i sum_i' P[i][i'] G[i'][i].  P == NULL means identity (E = Tr G). */
double sie_oracle_trace(int nocc, const double* P, const double* G) {
    long double e = 0.0L;
    for (int i = 0; i < nocc; ++i)
        for (int ip = 0; ip < nocc; ++ip) {
            double p = P ? P[(size_t)i * nocc + ip] : (i == ip ? 1.0 : 0.0);
            e += (long double)p * (long double)G[(size_t)ip * nocc + i];
        }
    return (double)e;
}

/*
 * NEXT-1: occupied block of the MP2 one-particle reduced density matrix, PAPER.md Eq. S18 (L357):
 *     gamma_ij = 2 delta_ij - 2 sum_k sum_ab t_ik^ab ( 2 t_jk^ab - t_jk^ba ),   t_ik^ab = (ia|kb) / (e_i + e_k - e_a - e_b)
 * (Eq. S15-S16, with the sign folded into the denominator as in O5; gamma is quadratic in t).
 *   B [nocc][nvir][naux], e_occ[nocc], e_vir[nvir]; gamma [nocc][nocc] row-major, OVERWRITTEN.
 * Loops in the paper's order: for each k, the amplitudes t_ik^ab of all i, then every (i, j) pair.  Returns 0, or 1 on
 * allocation failure.  Pins: tests/test_oracle_pins.py (closed form o=v=1, brute force from explicit four-index
 * amplitudes, gamma_ii = 2 + dE/de_i against the pinned energy, symmetry, positive semi-definiteness of 2 - gamma).
 */
int sie_oracle_rdm_occ(int nocc, int nvir, int naux, const double* B, const double* e_occ, const double* e_vir,
                       double* gamma) {
    const size_t vv = (size_t)nvir * nvir;
    double* Tk = (double*)malloc(sizeof(double) * (size_t)nocc * vv);      /* t_ik^ab for all i at fixed k */
    long double* Gl = (long double*)calloc((size_t)nocc * nocc, sizeof(long double));
    if (!Tk || !Gl) { free(Tk); free(Gl); return 1; }
    for (int k = 0; k < nocc; ++k) {
#pragma omp parallel for collapse(2) schedule(static)
        for (int i = 0; i < nocc; ++i)
            for (int a = 0; a < nvir; ++a) {
                const double* bia = B + ((size_t)i * nvir + a) * naux;
                double* t = Tk + (size_t)i * vv + (size_t)a * nvir;
                for (int b = 0; b < nvir; ++b)
                    t[b] = dot8(bia, B + ((size_t)k * nvir + b) * naux, naux) / (e_occ[i] + e_occ[k] - e_vir[a] - e_vir[b]);
            }
#pragma omp parallel for collapse(2) schedule(static)
        for (int i = 0; i < nocc; ++i)
            for (int j = 0; j < nocc; ++j) {
                const double* Ti = Tk + (size_t)i * vv;
                const double* Tj = Tk + (size_t)j * vv;
                long double s = 0.0L;
                for (int a = 0; a < nvir; ++a)
                    for (int b = 0; b < nvir; ++b)
                        s += (long double)Ti[(size_t)a * nvir + b] *
                             (2.0L * (long double)Tj[(size_t)a * nvir + b] - (long double)Tj[(size_t)b * nvir + a]);
                Gl[(size_t)i * nocc + j] += s;
            }
    }
    for (int i = 0; i < nocc; ++i)
        for (int j = 0; j < nocc; ++j)
            gamma[(size_t)i * nocc + j] = (double)((i == j ? 2.0L : 0.0L) - 2.0L * Gl[(size_t)i * nocc + j]);
    free(Tk);
    free(Gl);
    return 0;
}

/*
 * NEXT-1: virtual block of the MP2 one-particle reduced density matrix, PAPER.md Eq. S17 (L355):
 *     gamma_ab = 2 sum_ij sum_c t_ij^ac ( 2 t_ij^bc - t_ij^cb ),        t_ij^ac = (ia|jc) / (e_i + e_j - e_a - e_c)
 * (Eq. S15-S16; the sign of t cancels in the quadratic form).  The sub-space of Eq. S13-S14 (L338-L343) is
 * whatever orbital sets the caller put into B: impurity-occupied x environment-virtual for the virtual BNOs.
 *   B [nocc][nvir][naux], e_occ[nocc], e_vir[nvir]; gamma [nvir][nvir] row-major, OVERWRITTEN.
 * Loops in the paper's order: for each pair (i, j) the amplitude block t_ij^{ac} (nvir x nvir), then every (a, b) with the
 * sum over c; long-double accumulation.  Returns 0, or 1 on allocation failure.
 * Pins: tests/test_oracle_rdm_pins.py (closed form o=v=1, hand-worked case, brute force from explicit four-index amplitudes,
 * Tr gamma_occ + Tr gamma_vir = 2 nocc, gamma_aa = dE/de_a against the pinned energy, symmetry, positive semi-definiteness).
 */
int sie_oracle_rdm_vir(int nocc, int nvir, int naux, const double* B, const double* e_occ, const double* e_vir,
                       double* gamma) {
    const size_t vv = (size_t)nvir * nvir;
    double* T = (double*)malloc(sizeof(double) * vv);                      /* t_ij^ac for one (i, j) */
    long double* Gl = (long double*)calloc(vv, sizeof(long double));
    if (!T || !Gl) { free(T); free(Gl); return 1; }
    for (int i = 0; i < nocc; ++i)
        for (int j = 0; j < nocc; ++j) {
#pragma omp parallel for schedule(static)
            for (int a = 0; a < nvir; ++a) {
                const double* bia = B + ((size_t)i * nvir + a) * naux;
                for (int c = 0; c < nvir; ++c)
                    T[(size_t)a * nvir + c] =
                        dot8(bia, B + ((size_t)j * nvir + c) * naux, naux) / (e_occ[i] + e_occ[j] - e_vir[a] - e_vir[c]);
            }
#pragma omp parallel for collapse(2) schedule(static)
            for (int a = 0; a < nvir; ++a)
                for (int b = 0; b < nvir; ++b) {
                    long double s = 0.0L;
                    for (int c = 0; c < nvir; ++c)
                        s += (long double)T[(size_t)a * nvir + c] *
                             (2.0L * (long double)T[(size_t)b * nvir + c] - (long double)T[(size_t)c * nvir + b]);
                    Gl[(size_t)a * nvir + b] += s;
                }
        }
    for (size_t k = 0; k < vv; ++k) gamma[k] = (double)(2.0L * Gl[k]);
    free(T);
    free(Gl);
    return 0;
}
