/* ORACLE — TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU implementation of the Moebius/Shamir
 * domain-wall-fermion operator of arXiv:2203.17119's hot path, written from
 * the definitions (DESIGN.md §2 "readings") and the
 * paper's block algebra (eqs. 3-5, PAPER.md:175 Dirichlet
 * wrapper, "usual red-black preconditioned").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no
 * code, header, table or constant with paper_2203_17119_b200/csrc.
 *
 * Everything is written site-by-site with full 4x4 gamma matrices and full
 * 3x3 links (no half-spinor trick, no 2-row compression, no dense s-tables,
 * no blocking, no fusion).  Mooee^{-1} is the sequential s-sweep (C5), NOT
 * the closed-form table the CUDA path uses.
 *
 * Compile twice: -DORC_REAL=double -DORC_SUFFIX=_f64 and
 *                -DORC_REAL=float  -DORC_SUFFIX=_f32   (oracle/build.py).
 *
 * Canonical layouts (all arrays are C-contiguous ORC_REAL):
 *   gauge   [lex][mu][row][col][re,im],  lex = ((t*Lz+z)*Ly+y)*Lx+x,
 *           mu = 0..3 = x,y,z,t; U_mu(x) links x -> x+mu_hat
 *   FULL    [lex][s][spin][colour][re,im]
 *   EVEN/ODD[cb ][s][spin][colour][re,im],  cb = lex/2 over the sites with
 *           (x+y+z+t)%2 == parity (Lx is even so lex/2 enumerates them in order)
 */
#include <complex.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

#ifndef ORC_REAL
#define ORC_REAL double
#endif
#ifndef ORC_SUFFIX
#define ORC_SUFFIX _f64
#endif
#define ORC_CAT2(a, b) a##b
#define ORC_CAT(a, b) ORC_CAT2(a, b)
#define ORC(name) ORC_CAT(name, ORC_SUFFIX)

typedef ORC_REAL real;
typedef ORC_REAL _Complex cplx;

/* parameters: SURVEY §8(c) C2-C7 */
typedef struct {
    int L[4];           /* Lx, Ly, Lz, Lt (all even) */
    int Ls;
    double M5, mf, b5, c5;
    int antiperiodic_t; /* C2: factor -1 on the hop across t = Lt-1 -> 0 */
} orc_params;

/* ---- C1: chiral gamma basis, gamma5 = diag(1,1,-1,-1) ------------------ */
static const double _Complex GAMMA[4][4][4] = {
    /* gamma_x */ {{0, 0, 0, I}, {0, 0, I, 0}, {0, -I, 0, 0}, {-I, 0, 0, 0}},
    /* gamma_y */ {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    /* gamma_z */ {{0, 0, I, 0}, {0, 0, 0, -I}, {-I, 0, 0, 0}, {0, I, 0, 0}},
    /* gamma_t */ {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};

static inline long lex_of(const int L[4], const int x[4]) {
    return (((long)x[3] * L[2] + x[2]) * L[1] + x[1]) * L[0] + x[0];
}
static inline void coords_of(const int L[4], long lex, int x[4]) {
    x[0] = (int)(lex % L[0]); lex /= L[0];
    x[1] = (int)(lex % L[1]); lex /= L[1];
    x[2] = (int)(lex % L[2]); lex /= L[2];
    x[3] = (int)lex;
}
static inline long vol4(const orc_params* p) {
    return (long)p->L[0] * p->L[1] * p->L[2] * p->L[3];
}

/* ---- C7: Dirichlet cut (BCs applied to the gauge argument) --
 * cut[mu] = B > 0 zeroes U_mu(x) for every x with x_mu mod B == B-1
 * (including the periodic wrap link).                                       */
void ORC(orc_apply_cut)(const orc_params* p, const int cut[4], const real* Uin, real* Uout) {
    long V = vol4(p);
    memcpy(Uout, Uin, sizeof(real) * V * 4 * 18);
    for (long lex = 0; lex < V; ++lex) {
        int x[4];
        coords_of(p->L, lex, x);
        for (int mu = 0; mu < 4; ++mu) {
            int B = cut[mu];
            if (B > 0 && (x[mu] % B) == B - 1)
                for (int k = 0; k < 18; ++k) Uout[(lex * 4 + mu) * 18 + k] = 0;
        }
    }
}

/* ---- C3: Dhop ----------------------------------------------------------
 * Dhop psi(x,s) = sum_mu [ (1 - g_mu) U_mu(x) psi(x+mu,s)
 *                        + (1 + g_mu) U_mu(x-mu)^dag psi(x-mu,s) ]
 * dagger swaps the two projector signs.  No prefactor.
 * out_parity: 0 even, 1 odd (in = opposite-parity half field, out = half
 * field), 2 full (both FULL fields).                                        */
static inline long field_site(long lex, int parity_mode) {
    return parity_mode == 2 ? lex : lex / 2;
}

/* all Ls slices of one output site `lex`; osite = where the result goes in `out` */
static void dhop_site(const orc_params* p, const cplx* Uc, const cplx* in, cplx* out, long lex, long osite,
                      int out_parity, int dagger) {
    const int Ls = p->Ls;
    int x[4];
    coords_of(p->L, lex, x);
    for (int s = 0; s < Ls; ++s) {
        cplx acc[4][3];
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) acc[a][c] = 0;
        for (int mu = 0; mu < 4; ++mu) {
            for (int dir = 0; dir < 2; ++dir) { /* 0: forward leg, 1: backward leg */
                int y[4] = {x[0], x[1], x[2], x[3]};
                double bc = 1.0;
                if (dir == 0) {
                    y[mu] = (x[mu] + 1) % p->L[mu];
                    if (mu == 3 && p->antiperiodic_t && x[3] == p->L[3] - 1) bc = -1.0;
                } else {
                    y[mu] = (x[mu] - 1 + p->L[mu]) % p->L[mu];
                    if (mu == 3 && p->antiperiodic_t && x[3] == 0) bc = -1.0;
                }
                long ylex = lex_of(p->L, y);
                const cplx* link = Uc + ((dir == 0 ? lex : ylex) * 4 + mu) * 9;
                const cplx* psi = in + (field_site(ylex, out_parity) * Ls + s) * 12;
                /* colour multiply: chi[a][c] = sum_c' W[c][c'] psi[a][c'] */
                cplx chi[4][3];
                for (int a = 0; a < 4; ++a)
                    for (int c = 0; c < 3; ++c) {
                        cplx t = 0;
                        for (int cp = 0; cp < 3; ++cp) {
                            cplx w = (dir == 0) ? link[c * 3 + cp] : conj(link[cp * 3 + c]);
                            t += w * psi[a * 3 + cp];
                        }
                        chi[a][c] = (real)bc * t;
                    }
                /* spin: (1 -/+ gamma_mu), full 4x4 the slow way */
                double sg = (dir == 0) ? -1.0 : +1.0;
                if (dagger) sg = -sg;
                for (int a = 0; a < 4; ++a)
                    for (int c = 0; c < 3; ++c) {
                        cplx t = chi[a][c];
                        for (int b = 0; b < 4; ++b)
                            t += (cplx)(sg * GAMMA[mu][a][b]) * chi[b][c];
                        acc[a][c] += t;
                    }
            }
        }
        cplx* o = out + (osite * Ls + s) * 12;
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) o[a * 3 + c] = acc[a][c];
    }
}

void ORC(orc_dhop)(const orc_params* p, const real* U, const real* in_, real* out_,
                   int out_parity, int dagger) {
    const cplx* in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
    const cplx* Uc = (const cplx*)U;
    const long V = vol4(p);
#pragma omp parallel for schedule(static)
    for (long lex = 0; lex < V; ++lex) {
        int x[4];
        coords_of(p->L, lex, x);
        int par = (x[0] + x[1] + x[2] + x[3]) & 1;
        if (out_parity != 2 && par != out_parity) continue;
        dhop_site(p, Uc, in, out, lex, field_site(lex, out_parity), out_parity, dagger);
    }
}

/* ---- C4: s-hop Q and its adjoint ---------------------------------------
 * (Q psi)_s  = P_- psi_{s+1} + P_+ psi_{s-1},  psi_{Ls} = -mf psi_0,
 *                                              psi_{-1} = -mf psi_{Ls-1}
 * (Q^dag psi)_s = P_+ psi_{s+1} + P_- psi_{s-1}, same walls.
 * P_+ = spin rows 0,1; P_- = spin rows 2,3 (gamma5 = diag(1,1,-1,-1)).
 * n4 = number of 4-D sites in the field (V4 or V4/2).                       */
static void apply_Q(const orc_params* p, long n4, const cplx* in, cplx* out, int dagger) {
    const int Ls = p->Ls;
    const real mf = (real)p->mf;
#pragma omp parallel for schedule(static)
    for (long site = 0; site < n4; ++site)
        for (int s = 0; s < Ls; ++s)
            for (int a = 0; a < 4; ++a) {
                int upper = (a < 2);                 /* P_+ component */
                /* Q: P_+ takes s-1, P_- takes s+1;  Q^dag: P_+ takes s+1, P_- takes s-1 */
                int take_minus = dagger ? !upper : upper;
                int sp;
                real w = 1;
                if (take_minus) { sp = s - 1; if (sp < 0) { sp = Ls - 1; w = -mf; } }
                else            { sp = s + 1; if (sp >= Ls) { sp = 0; w = -mf; } }
                for (int c = 0; c < 3; ++c)
                    out[(site * Ls + s) * 12 + a * 3 + c] = w * in[(site * Ls + sp) * 12 + a * 3 + c];
            }
}

/* out = alpha*in + beta*Q(in)  (or Q^dag) */
static void apply_aQ(const orc_params* p, long n4, const real* in, real* out, double alpha, double beta, int dagger) {
    long n = n4 * p->Ls * 24;
    real* tmp = (real*)malloc(sizeof(real) * n);
    apply_Q(p, n4, (const cplx*)in, (cplx*)tmp, dagger);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) out[i] = (real)alpha * in[i] + (real)beta * tmp[i];
    free(tmp);
}

/* C5: A = b5 + c5 Q  ("Meooe5D") */
void ORC(orc_meooe5d)(const orc_params* p, long n4, const real* in, real* out, int dagger) {
    apply_aQ(p, n4, in, out, p->b5, p->c5, dagger);
}
/* C5: Mooee = bee - cee Q, bee = 1 + b5(4-M5), cee = 1 - c5(4-M5) */
void ORC(orc_mooee)(const orc_params* p, long n4, const real* in, real* out, int dagger) {
    double bee = 1.0 + p->b5 * (4.0 - p->M5), cee = 1.0 - p->c5 * (4.0 - p->M5);
    apply_aQ(p, n4, in, out, bee, -cee, dagger);
}

/* C5: Mooee^{-1} by the O(Ls) sequential sweep.
 * P_+ comps: z_s = (x_s + cee z_{s-1})/bee ascending, y_{Ls-1} = z_{Ls-1}/(1+mf r^Ls),
 *            y_s = z_s - mf r^{s+1} y_{Ls-1};
 * P_- comps mirror: z_s = (x_s + cee z_{s+1})/bee descending, y_0 = z_0/(1+mf r^Ls),
 *            y_s = z_s - mf r^{Ls-s} y_0.           r = cee/bee.
 * (Mooee^dag)^{-1} swaps the roles of the two chiralities.                  */
void ORC(orc_mooee_inv)(const orc_params* p, long n4, const real* in_, real* out_, int dagger) {
    const cplx* in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
    const int Ls = p->Ls;
    const double bee = 1.0 + p->b5 * (4.0 - p->M5), cee = 1.0 - p->c5 * (4.0 - p->M5);
    const double r = cee / bee;
    const double den = 1.0 + p->mf * pow(r, Ls);
#pragma omp parallel for schedule(static)
    for (long site = 0; site < n4; ++site) {
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) {
                int upper = (a < 2);
                int ascending = dagger ? !upper : upper;
                const long base = site * Ls * 12 + a * 3 + c;
                cplx z[64];
                if (ascending) {
                    cplx prev = 0;
                    for (int s = 0; s < Ls; ++s) { z[s] = (in[base + s * 12] + (real)cee * prev) / (real)bee; prev = z[s]; }
                    cplx yl = z[Ls - 1] / (real)den;
                    for (int s = 0; s < Ls - 1; ++s) out[base + s * 12] = z[s] - (real)(p->mf * pow(r, s + 1)) * yl;
                    out[base + (Ls - 1) * 12] = yl;
                } else {
                    cplx prev = 0;
                    for (int s = Ls - 1; s >= 0; --s) { z[s] = (in[base + s * 12] + (real)cee * prev) / (real)bee; prev = z[s]; }
                    cplx y0 = z[0] / (real)den;
                    for (int s = 1; s < Ls; ++s) out[base + s * 12] = z[s] - (real)(p->mf * pow(r, Ls - s)) * y0;
                    out[base] = y0;
                }
            }
    }
}

/* ---- C4: the full 5-D operator, straight from the definition -----------
 * D_W = (4-M5) - 1/2 Dhop;  M = (b5 D_W + 1) + (c5 D_W - 1) Q
 * M^dag = (b5 D_W^dag + 1) + Q^dag (c5 D_W^dag - 1)
 * FULL fields.                                                              */
static void apply_DW(const orc_params* p, const real* U, const real* in, real* out, int dagger) {
    long n = vol4(p) * p->Ls * 24;
    ORC(orc_dhop)(p, U, in, out, 2, dagger);
    real d = (real)(4.0 - p->M5);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) out[i] = d * in[i] - (real)0.5 * out[i];
}

void ORC(orc_M)(const orc_params* p, const real* U, const real* in, real* out, int dagger) {
    long V = vol4(p), n = V * p->Ls * 24;
    real* t1 = (real*)malloc(sizeof(real) * n);
    real* t2 = (real*)malloc(sizeof(real) * n);
    if (!dagger) {
        apply_Q(p, V, (const cplx*)in, (cplx*)t1, 0);      /* t1 = Q psi           */
        apply_DW(p, U, t1, t2, 0);                          /* t2 = D_W Q psi       */
        apply_DW(p, U, in, out, 0);                         /* out = D_W psi        */
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i)
            out[i] = (real)p->b5 * out[i] + in[i] + (real)p->c5 * t2[i] - t1[i];
    } else {
        apply_DW(p, U, in, t1, 1);                          /* t1 = D_W^dag psi     */
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) t2[i] = (real)p->c5 * t1[i] - in[i];   /* D_-^dag psi */
        apply_Q(p, V, (const cplx*)t2, (cplx*)out, 1);      /* out = Q^dag D_-^dag  */
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) out[i] += (real)p->b5 * t1[i] + in[i];
    }
    free(t1);
    free(t2);
}

/* ---- C5: Meooe = -1/2 Dhop A  (parity off-diagonal), half fields -------
 * out_parity is the parity of the OUTPUT; the input has the other parity.
 * dagger: (Meooe)^dag restricted to out_parity = -1/2 A^dag Dhop^dag.       */
void ORC(orc_meooe)(const orc_params* p, const real* U, const real* in, real* out, int out_parity, int dagger) {
    long n4 = vol4(p) / 2, n = n4 * p->Ls * 24;
    real* t = (real*)malloc(sizeof(real) * n);
    if (!dagger) {
        ORC(orc_meooe5d)(p, n4, in, t, 0);
        ORC(orc_dhop)(p, U, t, out, out_parity, 0);
    } else {
        ORC(orc_dhop)(p, U, in, t, out_parity, 1);
        ORC(orc_meooe5d)(p, n4, t, out, 1);
    }
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) out[i] *= (real)(-0.5);
    free(t);
}

/* ---- C6: Schur operator on the ODD sites ("usual red-black") --
 * Mpc = Moo - Moe Mee^{-1} Meo;  Mpc^dag = Moo^dag - Meo^dag Mee^{-dag} Moe^dag */
void ORC(orc_mpc)(const orc_params* p, const real* U, const real* in, real* out, int dagger) {
    long n4 = vol4(p) / 2, n = n4 * p->Ls * 24;
    real* t1 = (real*)malloc(sizeof(real) * n);
    real* t2 = (real*)malloc(sizeof(real) * n);
    if (!dagger) {
        ORC(orc_meooe)(p, U, in, t1, 0, 0);        /* Meo psi_o        (even) */
        ORC(orc_mooee_inv)(p, n4, t1, t2, 0);      /* Mee^{-1} ...     (even) */
        ORC(orc_meooe)(p, U, t2, t1, 1, 0);        /* Moe ...          (odd)  */
    } else {
        /* Moe^dag maps odd -> even: it is the dagger of the odd<-even hop, output parity even */
        ORC(orc_meooe)(p, U, in, t1, 0, 1);
        ORC(orc_mooee_inv)(p, n4, t1, t2, 1);
        ORC(orc_meooe)(p, U, t2, t1, 1, 1);
    }
    ORC(orc_mooee)(p, n4, in, out, dagger);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) out[i] -= t1[i];
    free(t1);
    free(t2);
}

void ORC(orc_mdagm)(const orc_params* p, const real* U, const real* in, real* out) {
    long n = vol4(p) / 2 * p->Ls * 24;
    real* t = (real*)malloc(sizeof(real) * n);
    ORC(orc_mpc)(p, U, in, t, 0);
    ORC(orc_mpc)(p, U, t, out, 1);
    free(t);
}

/* sum |v_i|^2 accumulated in double regardless of ORC_REAL (C8: reductions in fp64) */
double ORC(orc_norm2)(const real* v, long n) {
    double acc = 0;
#pragma omp parallel for schedule(static) reduction(+ : acc)
    for (long i = 0; i < n; ++i) acc += (double)v[i] * (double)v[i];
    return acc;
}

int ORC(orc_sizeof_real)(void) { return (int)sizeof(real); }

/* the gamma table in use, for the Clifford-algebra pin: out[a][b][re,im] as doubles */
void ORC(orc_gamma)(int mu, double* out) {
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) {
            out[(a * 4 + b) * 2 + 0] = creal(GAMMA[mu][a][b]);
            out[(a * 4 + b) * 2 + 1] = cimag(GAMMA[mu][a][b]);
        }
}
