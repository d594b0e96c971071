/*
 * hirep_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, literal evaluation of the Wilson-Dirac operator for fermions in a representation R
 * of SU(N_g), written from the text of arXiv 2503.06721.  It is the parity target for the
 * CUDA library and the timed "cpu_baseline" of bench.py.  It shares NO code with the CUDA path
 * (no headers, tables, helpers); only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  Everything is double precision, canonical lexicographic layout:
 *
 *     ix = ((t*L + x)*L + y)*L + z ;  spinor[ix][spin][colour] ;  links[ix][mu][row][col] (row-major)
 *
 * What follows the paper literally:
 *   - Pauli matrices Eq 1 (L173), e_mu Eq 2 (L178), gamma_mu Eq 3 (L182) as full 4x4 matrices;
 *     gamma_5 := gamma_0 gamma_1 gamma_2 gamma_3 (reading A1 of DESIGN.md; the paper never defines it).
 *   - D_m Eq 8 (L207) with a = 1 (reading A2):  (4+m) psi(x) - 1/2 sum_mu [ (1-gamma_mu) (x) U^R_mu(x) psi(x+mu)
 *     + (1+gamma_mu) (x) U^R_mu(x-mu)^dagger psi(x-mu) ], the (1 -+ gamma_mu) (x) U products formed as explicit
 *     Kronecker-structured sums -- no spin projection trick.
 *   - Boundary conditions: literal Eq 58/61 (L930-938): a hop that crosses the lattice boundary in direction mu
 *     picks up bc[mu] = +1 (periodic) or -1 (antiperiodic).  NOT the link-sign implementation of L945.
 *   - even/odd: (t+x+y+z) mod 2 (L793); block operators Eq 41 (L795); D_hat Eq 44 (L808); Q = g5 D Eq 11 (L230).
 *   - represented links (Eq 7; construction deferred by the paper to its ref [26]) from dense basis
 *     matrices by trace formulas (readings A10, A11 of DESIGN.md):
 *        ADJ  R_ab = 2 Re tr(T^a U T^b U^dagger),  tr(T^a T^b) = delta_ab/2  (T_FUND = 1/2, Tbl 1 L215)
 *        SYM / 2AS  R_AB = tr[(e^A)^T U e^B U^T]  over an orthonormal basis of (anti)symmetric N x N matrices.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): gamma algebra; free-field plane-wave closed forms;
 * gamma_5-hermiticity; gauge covariance; representation homomorphism / unitarity / d_R / T_R / textbook SU(2)
 * adjoint rotation / 2x2 minors; independent numpy dense-matrix assembly on 4^4 (oracle/dense.py) with the
 * block identities Eq 41-44; BC-as-link-sign equivalence.  Basis conventions (sign of gamma_5, generator and
 * tensor basis order) are not fixed by the paper and are "parity unpinned" by it; they are fixed in DESIGN.md.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -std=c11 -o liboracle.so hirep_oracle.c -lm
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

enum { REP_FUND = 0, REP_ADJ = 1, REP_SYM = 2, REP_ASY = 3 };

/* ------------------------------------------------------------------ gamma matrices (Eq 1-3) */
/* g[mu] is the 4x4 matrix gamma_mu, row-major g[mu][4*a+b]. */
void oracle_gamma(cplx *g /* [4][16] */) {
    cplx sigma[4][2][2];
    /* sigma[0] unused slot holds the 2x2 identity for e_0 */
    sigma[0][0][0] = 1; sigma[0][0][1] = 0; sigma[0][1][0] = 0; sigma[0][1][1] = 1;
    sigma[1][0][0] = 0; sigma[1][0][1] = 1; sigma[1][1][0] = 1; sigma[1][1][1] = 0;          /* Eq 1 */
    sigma[2][0][0] = 0; sigma[2][0][1] = -I; sigma[2][1][0] = I; sigma[2][1][1] = 0;
    sigma[3][0][0] = 1; sigma[3][0][1] = 0; sigma[3][1][0] = 0; sigma[3][1][1] = -1;
    for (int mu = 0; mu < 4; ++mu) {
        cplx e[2][2];
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                e[a][b] = (mu == 0) ? -sigma[0][a][b] : -I * sigma[mu][a][b];                  /* Eq 2 */
        cplx *G = g + 16 * mu;
        for (int k = 0; k < 16; ++k) G[k] = 0;
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b) {
                G[4 * a + (2 + b)] = e[a][b];                 /* upper right block  e_mu          */
                G[4 * (2 + a) + b] = conj(e[b][a]);           /* lower left block   e_mu^dagger   Eq 3 */
            }
    }
}

static void mat4_mul(const cplx *A, const cplx *B, cplx *C) {
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) {
            cplx s = 0;
            for (int c = 0; c < 4; ++c) s += A[4 * a + c] * B[4 * c + b];
            C[4 * a + b] = s;
        }
}

/* gamma_5 = gamma_0 gamma_1 gamma_2 gamma_3 */
void oracle_gamma5(cplx *g5 /* [16] */) {
    cplx g[64], t1[16], t2[16];
    oracle_gamma(g);
    mat4_mul(g, g + 16, t1);
    mat4_mul(t1, g + 32, t2);
    mat4_mul(t2, g + 48, g5);
}

/* ------------------------------------------------------------- representations (Tbl 1, Eq 7) */
int oracle_rep_dim(int N, int rep) {
    switch (rep) {
    case REP_FUND: return N;
    case REP_ADJ: return N * N - 1;
    case REP_SYM: return N * (N + 1) / 2;
    case REP_ASY: return N * (N - 1) / 2;
    }
    return -1;
}

/* Generators of su(N), tr(T^a T^b) = delta_ab / 2, generalised Gell-Mann matrices ordered (reading A10):
 *   for j = 1..N-1 { for i = 0..j-1 { S_ij = (E_ij + E_ji)/2 ,  A_ij = -i (E_ij - E_ji)/2 } ,
 *                    D_j = diag(1,..,1 (j times), -j, 0,..) / sqrt(2 j (j+1)) }
 * which gives sigma_{1,2,3}/2 for N = 2 and lambda_{1..8}/2 for N = 3.   Tgen[a][N*N], a = 0..N*N-2. */
void oracle_generators(int N, cplx *Tgen) {
    int a = 0;
    memset(Tgen, 0, sizeof(cplx) * (size_t)(N * N - 1) * N * N);
    for (int j = 1; j < N; ++j) {
        for (int i = 0; i < j; ++i) {
            cplx *S = Tgen + (size_t)a * N * N; ++a;
            S[i * N + j] = 0.5; S[j * N + i] = 0.5;
            cplx *A = Tgen + (size_t)a * N * N; ++a;
            A[i * N + j] = -0.5 * I; A[j * N + i] = 0.5 * I;
        }
        cplx *D = Tgen + (size_t)a * N * N; ++a;
        double nrm = 1.0 / sqrt(2.0 * j * (j + 1));
        for (int k = 0; k < j; ++k) D[k * N + k] = nrm;
        D[j * N + j] = -j * nrm;
    }
}

/* Orthonormal real basis of 2-index tensors (reading A11): pairs (i,j) in lexicographic order,
 *   2AS: i<j, (E_ij - E_ji)/sqrt2 ;   SYM: i<=j, E_ii  or (E_ij + E_ji)/sqrt2 .     B[A][N*N] */
void oracle_tensor_basis(int N, int rep, double *B) {
    int A = 0, d = oracle_rep_dim(N, rep);
    memset(B, 0, sizeof(double) * (size_t)d * N * N);
    const double r = 1.0 / sqrt(2.0);
    for (int i = 0; i < N; ++i)
        for (int j = i; j < N; ++j) {
            if (rep == REP_ASY) {
                if (i == j) continue;
                B[(size_t)A * N * N + i * N + j] = r;
                B[(size_t)A * N * N + j * N + i] = -r;
            } else {
                if (i == j) B[(size_t)A * N * N + i * N + i] = 1.0;
                else { B[(size_t)A * N * N + i * N + j] = r; B[(size_t)A * N * N + j * N + i] = r; }
            }
            ++A;
        }
}

static void matN_mul(int N, const cplx *A, const cplx *B, cplx *C) {
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) {
            cplx s = 0;
            for (int k = 0; k < N; ++k) s += A[i * N + k] * B[k * N + j];
            C[i * N + j] = s;
        }
}

/* R[dR*dR] (row-major, complex; the adjoint comes out with zero imaginary part) from U[N*N]. */
int oracle_rep_matrix(int N, int rep, const cplx *U, cplx *R) {
    const int d = oracle_rep_dim(N, rep);
    if (d < 0) return -1;
    if (rep == REP_FUND) { memcpy(R, U, sizeof(cplx) * N * N); return 0; }
    cplx *t1 = malloc(sizeof(cplx) * N * N), *t2 = malloc(sizeof(cplx) * N * N), *t3 = malloc(sizeof(cplx) * N * N);
    cplx *X = malloc(sizeof(cplx) * N * N);
    if (rep == REP_ADJ) {
        cplx *Tg = malloc(sizeof(cplx) * (size_t)d * N * N);
        oracle_generators(N, Tg);
        for (int i = 0; i < N; ++i) for (int j = 0; j < N; ++j) X[i * N + j] = conj(U[j * N + i]);   /* U^dagger */
        for (int a = 0; a < d; ++a)
            for (int b = 0; b < d; ++b) {
                matN_mul(N, Tg + (size_t)a * N * N, U, t1);          /* T^a U               */
                matN_mul(N, t1, Tg + (size_t)b * N * N, t2);         /* T^a U T^b           */
                matN_mul(N, t2, X, t3);                              /* T^a U T^b U^dagger  */
                cplx tr = 0;
                for (int k = 0; k < N; ++k) tr += t3[k * N + k];
                R[a * d + b] = 2.0 * creal(tr);
            }
        free(Tg);
    } else {
        double *B = malloc(sizeof(double) * (size_t)d * N * N);
        cplx *EA = malloc(sizeof(cplx) * N * N), *EB = malloc(sizeof(cplx) * N * N);
        oracle_tensor_basis(N, rep, B);
        for (int i = 0; i < N; ++i) for (int j = 0; j < N; ++j) X[i * N + j] = U[j * N + i];          /* U^T */
        for (int a = 0; a < d; ++a)
            for (int b = 0; b < d; ++b) {
                for (int i = 0; i < N; ++i) for (int j = 0; j < N; ++j) {
                    EA[i * N + j] = B[(size_t)a * N * N + j * N + i];                                  /* (e^A)^T */
                    EB[i * N + j] = B[(size_t)b * N * N + i * N + j];
                }
                matN_mul(N, EA, U, t1);                              /* (e^A)^T U           */
                matN_mul(N, t1, EB, t2);                             /* (e^A)^T U e^B       */
                matN_mul(N, t2, X, t3);                              /* (e^A)^T U e^B U^T   */
                cplx tr = 0;
                for (int k = 0; k < N; ++k) tr += t3[k * N + k];
                R[a * d + b] = tr;
            }
        free(B); free(EA); free(EB);
    }
    free(t1); free(t2); free(t3); free(X);
    return 0;
}

/* Represent a whole canonical gauge field: Rlinks[n][dR*dR] from links[n][N*N]. */
int oracle_represent_field(int N, int rep, long n_links, const cplx *links, cplx *Rlinks) {
    const int d = oracle_rep_dim(N, rep);
    if (d < 0) return -1;
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n_links; ++k)
        oracle_rep_matrix(N, rep, links + (size_t)k * N * N, Rlinks + (size_t)k * d * d);
    return 0;
}

/* --------------------------------------------------------------------- the hopping term, one site */
/* out[4*dR] = -1/2 sum_mu [ sf[mu] (1 - gamma_mu) (x) Rf[mu] psi_f[mu]  +  sb[mu] (1 + gamma_mu) (x) Rb[mu]^dagger psi_b[mu] ]
 *   Rf[mu] = U^R_mu(x), psi_f[mu] = psi(x+mu);  Rb[mu] = U^R_mu(x-mu), psi_b[mu] = psi(x-mu);
 *   sf/sb = boundary factor of that hop (Eq 61).  Pointer arrays index mu = 0..3.                 (Eq 8) */
void oracle_hop_local(int dR, const cplx *const *Rf, const cplx *const *Rb, const cplx *const *psi_f,
                      const cplx *const *psi_b, const double *sf, const double *sb, cplx *out) {
    cplx g[64];
    oracle_gamma(g);
    for (int k = 0; k < 4 * dR; ++k) out[k] = 0;
    for (int mu = 0; mu < 4; ++mu) {
        const cplx *G = g + 16 * mu;
        for (int al = 0; al < 4; ++al)
            for (int be = 0; be < 4; ++be) {
                const cplx Pm = ((al == be) ? 1.0 : 0.0) - G[4 * al + be];   /* (1 - gamma_mu)_{al,be} */
                const cplx Pp = ((al == be) ? 1.0 : 0.0) + G[4 * al + be];   /* (1 + gamma_mu)_{al,be} */
                for (int i = 0; i < dR; ++i) {
                    cplx accf = 0, accb = 0;
                    for (int j = 0; j < dR; ++j) {
                        accf += Rf[mu][i * dR + j] * psi_f[mu][be * dR + j];
                        accb += conj(Rb[mu][j * dR + i]) * psi_b[mu][be * dR + j];   /* (R^dagger)_ij */
                    }
                    out[al * dR + i] += -0.5 * (sf[mu] * Pm * accf + sb[mu] * Pp * accb);
                }
            }
    }
}

/* ----------------------------------------------------------------------------- full-lattice fields */
static inline long site_index(int L, int t, int x, int y, int z) { return (((long)t * L + x) * L + y) * L + z; }

/* hop(psi) on every site of a T x L^3 lattice.  Rlinks[ix][mu][dR*dR], psi/out [ix][4*dR]. */
void oracle_hop_field(int T, int L, int dR, const int *bc, const cplx *Rlinks, const cplx *psi, cplx *out) {
    const int ext[4] = {T, L, L, L};
    const size_t S = 4 * (size_t)dR, K = (size_t)dR * dR;
#pragma omp parallel for collapse(2) schedule(static)
    for (int t = 0; t < T; ++t)
        for (int x = 0; x < L; ++x)
            for (int y = 0; y < L; ++y)
                for (int z = 0; z < L; ++z) {
                    const int c[4] = {t, x, y, z};
                    const long ix = site_index(L, t, x, y, z);
                    const cplx *Rf[4], *Rb[4], *pf[4], *pb[4];
                    double sf[4], sb[4];
                    for (int mu = 0; mu < 4; ++mu) {
                        int cf[4] = {t, x, y, z}, cb[4] = {t, x, y, z};
                        cf[mu] = c[mu] + 1; sf[mu] = 1.0;
                        if (cf[mu] == ext[mu]) { cf[mu] = 0; sf[mu] = bc[mu]; }               /* Eq 58 / 61 */
                        cb[mu] = c[mu] - 1; sb[mu] = 1.0;
                        if (cb[mu] < 0) { cb[mu] = ext[mu] - 1; sb[mu] = bc[mu]; }
                        const long ixf = site_index(L, cf[0], cf[1], cf[2], cf[3]);
                        const long ixb = site_index(L, cb[0], cb[1], cb[2], cb[3]);
                        Rf[mu] = Rlinks + ((size_t)ix * 4 + mu) * K;
                        Rb[mu] = Rlinks + ((size_t)ixb * 4 + mu) * K;
                        pf[mu] = psi + (size_t)ixf * S;
                        pb[mu] = psi + (size_t)ixb * S;
                    }
                    oracle_hop_local(dR, Rf, Rb, pf, pb, sf, sb, out + (size_t)ix * S);
                }
}

/* D_m psi = (4+m) psi + hop(psi)                                                       (Eq 8, Eq 10) */
void oracle_Dphi(int T, int L, int dR, const int *bc, double m0, const cplx *Rlinks, const cplx *psi, cplx *out) {
    const size_t n = (size_t)T * L * L * L * 4 * dR;
    oracle_hop_field(T, L, dR, bc, Rlinks, psi, out);
    for (size_t k = 0; k < n; ++k) out[k] += (4.0 + m0) * psi[k];
}

static int site_parity(int L, long ix) {
    int z = ix % L, y = (ix / L) % L, x = (ix / ((long)L * L)) % L, t = ix / ((long)L * L * L);
    return (t + x + y + z) & 1;                                                             /* L793 */
}

/* Off-diagonal block of Eq 41: input lives on the sites of parity `pin` (listed in increasing ix),
 * output on the sites of parity 1-pin.  Done literally: embed in a full field that is zero on the other
 * parity, apply hop, restrict.  Dphi_eo: pin = 1 (odd in, even out); Dphi_oe: pin = 0.   (reading A3, A5) */
void oracle_Dphi_offdiag(int T, int L, int dR, const int *bc, int pin, const cplx *Rlinks, const cplx *psi_half,
                         cplx *out_half) {
    const long V = (long)T * L * L * L;
    const size_t S = 4 * (size_t)dR;
    cplx *full = calloc((size_t)V * S, sizeof(cplx)), *res = malloc((size_t)V * S * sizeof(cplx));
    long k = 0;
    for (long ix = 0; ix < V; ++ix)
        if (site_parity(L, ix) == pin) { memcpy(full + (size_t)ix * S, psi_half + (size_t)k * S, S * sizeof(cplx)); ++k; }
    oracle_hop_field(T, L, dR, bc, Rlinks, full, res);
    k = 0;
    for (long ix = 0; ix < V; ++ix)
        if (site_parity(L, ix) != pin) { memcpy(out_half + (size_t)k * S, res + (size_t)ix * S, S * sizeof(cplx)); ++k; }
    free(full); free(res);
}

/* D_hat psi_e = (4+m)^2 psi_e - D_eo D_oe psi_e                                              (Eq 44) */
void oracle_Dphi_hat(int T, int L, int dR, const int *bc, double m0, const cplx *Rlinks, const cplx *psi_e, cplx *out_e) {
    const size_t n = (size_t)T * L * L * L / 2 * 4 * dR;
    cplx *tmp_o = malloc(n * sizeof(cplx));
    oracle_Dphi_offdiag(T, L, dR, bc, 0, Rlinks, psi_e, tmp_o);      /* D_oe psi_e  (odd)  */
    oracle_Dphi_offdiag(T, L, dR, bc, 1, Rlinks, tmp_o, out_e);      /* D_eo (...)  (even) */
    for (size_t k = 0; k < n; ++k) out_e[k] = (4.0 + m0) * (4.0 + m0) * psi_e[k] - out_e[k];
    free(tmp_o);
}

/* apply gamma_5 (as a 4x4 matrix product) to every site */
void oracle_g5(long nsites, int dR, const cplx *in, cplx *out) {
    cplx g5[16];
    oracle_gamma5(g5);
    for (long s = 0; s < nsites; ++s)
        for (int al = 0; al < 4; ++al)
            for (int i = 0; i < dR; ++i) {
                cplx acc = 0;
                for (int be = 0; be < 4; ++be) acc += g5[4 * al + be] * in[((size_t)s * 4 + be) * dR + i];
                out[((size_t)s * 4 + al) * dR + i] = acc;
            }
}

/* Q_m^2 psi = gamma_5 D_m gamma_5 D_m psi                                             (Eq 11) */
void oracle_g5Dphi_sq(int T, int L, int dR, const int *bc, double m0, const cplx *Rlinks, const cplx *psi, cplx *out) {
    const long V = (long)T * L * L * L;
    const size_t n = (size_t)V * 4 * dR;
    cplx *a = malloc(n * sizeof(cplx)), *b = malloc(n * sizeof(cplx));
    oracle_Dphi(T, L, dR, bc, m0, Rlinks, psi, a);
    oracle_g5(V, dR, a, b);
    oracle_Dphi(T, L, dR, bc, m0, Rlinks, b, a);
    oracle_g5(V, dR, a, out);
    free(a); free(b);
}

int oracle_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
