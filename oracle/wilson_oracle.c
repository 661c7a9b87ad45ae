/*
 * wilson_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation of the Wilson hopping
 * operator ("dslash") and the fermion matrix built on it, written from the
 * definitions only.  It shares no code, header, table or helper with the CUDA
 * path under paper_1112_5280_b200/ and must never be imported, linked or
 * executed by it.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may use it.
 *
 * What the paper says (PAPER.md = /root/reference/PAPER.md at survey time):
 *   - PAPER.md:61  (sec. 3)  "N_f = 2 twisted-mass Wilson fermions", "even-odd preconditioning"
 *   - PAPER.md:89  (sec. 3)  "the non-diagonal part of the Dirac matrix ('dslash')"
 *   - PAPER.md:109 (sec. 4)  "M is the fermion matrix"
 * The paper prints no formula for the operator; the definition below is the
 * textbook Wilson form fixed in SURVEY.md sec. 8(c) / Appendix A (readings A1-A9):
 *
 *   (H psi)(x) = sum_{mu=0..3} [ (1 - gamma_mu) U_mu(x)        psi(x + mu^)
 *                              + (1 + gamma_mu) U_mu(x - mu^)^+ psi(x - mu^) ]
 *   M_full = 1 - kappa H
 *   parity p(x) = (x0+x1+x2+x3) mod 2,  H = [[0,H_eo],[H_oe,0]],  M_eo = 1 - kappa^2 H_eo H_oe  (even sites)
 *   boundary:  psi(x + L_mu mu^) = bc_mu psi(x), |bc_mu| = 1; the forward hop from x_mu = L_mu-1
 *              multiplies the neighbour by bc_mu, the backward hop from x_mu = 0 by conj(bc_mu);
 *              links are periodic and carry no phase (reading A6).
 *
 * Method: per output site, loop over mu, explicit (x +- 1 + L) % L neighbour
 * coordinates, w = U psi (or U^+ psi) per spin, then out += (1 -+ gamma_mu) w with
 * DENSE 4x4 complex gamma matrices from the table below (Appendix A.2).  No
 * half-spinor trick, no blocking, no reordering.  All arithmetic is fp64
 * (C99 double complex); inputs may be given as complex64 and are promoted
 * element by element (reading A14).
 *
 * Canonical layout (Appendix A.4), C-contiguous, complex interleaved:
 *   spinor [T][Z][Y][X][spin 4][colour 3]
 *   links  [mu 4][T][Z][Y][X][row 3][col 3],  (U psi)_a = sum_b U[a][b] psi_b,  U_mu(x) stored at x.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 plane waves, P2 free-field
 * spectrum on 4^4 (dense matrix), P3 gamma5-hermiticity, P4 even-odd == full,
 * P5 gauge covariance, P6 constant field, P7 point source written out by hand,
 * P8 Clifford algebra / projectors, P9 two-row reconstruction, P10 independent
 * numpy.roll formulation (oracle/roll_formulation.py), P11 linearity/translation; twisted-mass operator
 * (next row f1): T1 mu = 0 reduces to apply_M, T2 free-field plane waves, T3 gamma5 M(mu) gamma5 = M(-mu)^dagger,
 * T4 even-odd form = Schur complement of the full operator.
 * Parity unpinned: nothing.
 */
#include <complex.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* Appendix A.2: chiral basis, Hermitian, {g_mu,g_nu} = 2 delta, gamma5 = g_t g_x g_y g_z = diag(1,1,-1,-1). */
static const cplx GAMMA[5][4][4] = {
    /* gamma_x */
    {{0, 0, 0, -I},
     {0, 0, -I, 0},
     {0, I, 0, 0},
     {I, 0, 0, 0}},
    /* gamma_y */
    {{0, 0, 0, -1},
     {0, 0, 1, 0},
     {0, 1, 0, 0},
     {-1, 0, 0, 0}},
    /* gamma_z */
    {{0, 0, -I, 0},
     {0, 0, 0, I},
     {I, 0, 0, 0},
     {0, -I, 0, 0}},
    /* gamma_t */
    {{0, 0, -1, 0},
     {0, 0, 0, -1},
     {-1, 0, 0, 0},
     {0, -1, 0, 0}},
    /* gamma_5 */
    {{1, 0, 0, 0},
     {0, 1, 0, 0},
     {0, 0, -1, 0},
     {0, 0, 0, -1}},
};

typedef struct {
    const void *U;
    const void *psi;
    int u_f32;   /* 1: U is complex64, 0: complex128 */
    int psi_f32; /* same for psi */
    int L[4];    /* X, Y, Z, T */
    cplx bc[4];
} fields_t;

static inline size_t lex(const int L[4], const int x[4]) {
    return (size_t)x[0] + (size_t)L[0] * ((size_t)x[1] + (size_t)L[1] * ((size_t)x[2] + (size_t)L[2] * (size_t)x[3]));
}

static inline cplx ld(const void *base, size_t idx, int f32) {
    return f32 ? (cplx)((const float complex *)base)[idx] : ((const double complex *)base)[idx];
}

static inline cplx link(const fields_t *f, int mu, const int x[4], int a, int b) {
    size_t vol = (size_t)f->L[0] * f->L[1] * f->L[2] * f->L[3];
    return ld(f->U, (((size_t)mu * vol + lex(f->L, x)) * 3 + a) * 3 + b, f->u_f32);
}

static inline cplx spinor(const fields_t *f, const int x[4], int s, int c) {
    return ld(f->psi, (lex(f->L, x) * 4 + s) * 3 + c, f->psi_f32);
}

/* out[s][a] = (H psi)(x).  If nbr != NULL, nbr[2*mu+0] replaces psi(x+mu^) and nbr[2*mu+1] replaces
 * psi(x-mu^) (used to chain two hops at sampled sites); boundary phases are still applied here. */
static void hop_site(cplx out[4][3], const fields_t *f, const int x[4], cplx (*nbr)[4][3]) {
    for (int s = 0; s < 4; ++s)
        for (int a = 0; a < 3; ++a) out[s][a] = 0;

    for (int mu = 0; mu < 4; ++mu) {
        int xn[4] = {x[0], x[1], x[2], x[3]};
        cplx phi[4][3], w[4][3];

        /* forward: (1 - gamma_mu) U_mu(x) psi(x + mu^) */
        xn[mu] = (x[mu] + 1 + f->L[mu]) % f->L[mu];
        cplx phase = (x[mu] + 1 == f->L[mu]) ? f->bc[mu] : 1.0;
        for (int s = 0; s < 4; ++s)
            for (int c = 0; c < 3; ++c) phi[s][c] = phase * (nbr ? nbr[2 * mu][s][c] : spinor(f, xn, s, c));
        for (int s = 0; s < 4; ++s)
            for (int a = 0; a < 3; ++a) {
                cplx acc = 0;
                for (int b = 0; b < 3; ++b) acc += link(f, mu, x, a, b) * phi[s][b];
                w[s][a] = acc;
            }
        for (int s = 0; s < 4; ++s)
            for (int a = 0; a < 3; ++a) {
                cplx g = 0;
                for (int sp = 0; sp < 4; ++sp) g += GAMMA[mu][s][sp] * w[sp][a];
                out[s][a] += w[s][a] - g;
            }

        /* backward: (1 + gamma_mu) U_mu(x - mu^)^dagger psi(x - mu^) */
        xn[mu] = (x[mu] - 1 + f->L[mu]) % f->L[mu];
        phase = (x[mu] == 0) ? conj(f->bc[mu]) : 1.0;
        for (int s = 0; s < 4; ++s)
            for (int c = 0; c < 3; ++c) phi[s][c] = phase * (nbr ? nbr[2 * mu + 1][s][c] : spinor(f, xn, s, c));
        for (int s = 0; s < 4; ++s)
            for (int a = 0; a < 3; ++a) {
                cplx acc = 0;
                for (int b = 0; b < 3; ++b) acc += conj(link(f, mu, xn, b, a)) * phi[s][b];
                w[s][a] = acc;
            }
        for (int s = 0; s < 4; ++s)
            for (int a = 0; a < 3; ++a) {
                cplx g = 0;
                for (int sp = 0; sp < 4; ++sp) g += GAMMA[mu][s][sp] * w[sp][a];
                out[s][a] += w[s][a] + g;
            }
    }
}

static int setup(fields_t *f, const void *U, int u_f32, const void *psi, int psi_f32, const int dims[4],
                 const double bc_re[4], const double bc_im[4]) {
    if (!U || !psi || !dims || !bc_re || !bc_im) return 1;
    f->U = U;
    f->psi = psi;
    f->u_f32 = u_f32;
    f->psi_f32 = psi_f32;
    for (int mu = 0; mu < 4; ++mu) {
        if (dims[mu] < 2) return 1;
        f->L[mu] = dims[mu];
        f->bc[mu] = bc_re[mu] + I * bc_im[mu];
    }
    return 0;
}

/* mode: -1 all sites; 0/1 only output sites of that parity (others written as zero). */
static void hop_field(cplx *out, const fields_t *f, int mode) {
    const int X = f->L[0], Y = f->L[1], Z = f->L[2], T = f->L[3];
    const long vol = (long)X * Y * Z * T;
#pragma omp parallel for schedule(static)
    for (long n = 0; n < vol; ++n) {
        int x[4];
        long r = n;
        x[0] = (int)(r % X); r /= X;
        x[1] = (int)(r % Y); r /= Y;
        x[2] = (int)(r % Z); r /= Z;
        x[3] = (int)r;
        cplx(*o)[3] = (cplx(*)[3])(out + (size_t)n * 12);
        if (mode >= 0 && ((x[0] + x[1] + x[2] + x[3]) & 1) != mode) {
            for (int k = 0; k < 4; ++k)
                for (int a = 0; a < 3; ++a) o[k][a] = 0;
            continue;
        }
        hop_site(o, f, x, NULL);
    }
}

/* ------------------------------------------------------------------ exported API ---- */

/* mu = 0..3: gamma_mu; mu = 4: gamma_5.  out: 16 complex (row-major 4x4). */
void oracle_gamma(int mu, double complex *out) {
    for (int s = 0; s < 4; ++s)
        for (int t = 0; t < 4; ++t) out[4 * s + t] = GAMMA[mu][s][t];
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* out = H psi on every site.  out: complex128 [T][Z][Y][X][4][3]. */
int oracle_dslash_full(double complex *out, const void *U, int u_f32, const void *psi, int psi_f32,
                       const int dims[4], const double bc_re[4], const double bc_im[4]) {
    fields_t f;
    if (!out || setup(&f, U, u_f32, psi, psi_f32, dims, bc_re, bc_im)) return 1;
    hop_field(out, &f, -1);
    return 0;
}

/* out_p = H_{p,1-p} psi_{1-p}: written at sites of parity out_parity, zero elsewhere.
 * Reads psi only at sites of the other parity (all neighbours of a site have opposite parity). */
int oracle_dslash_eo(double complex *out, const void *U, int u_f32, const void *psi, int psi_f32,
                     const int dims[4], const double bc_re[4], const double bc_im[4], int out_parity) {
    fields_t f;
    if (!out || (out_parity != 0 && out_parity != 1)) return 1;
    if (setup(&f, U, u_f32, psi, psi_f32, dims, bc_re, bc_im)) return 1;
    for (int mu = 0; mu < 4; ++mu)
        if (dims[mu] & 1) return 1; /* checkerboarding needs even extents */
    hop_field(out, &f, out_parity);
    return 0;
}

/* eo = 0: out = psi - kappa H psi (all sites).
 * eo = 1: out_e = psi_e - kappa^2 H_eo H_oe psi_e on even sites, zero on odd sites (reading A8). */
int oracle_apply_M(double complex *out, const void *U, int u_f32, const void *psi, int psi_f32,
                   const int dims[4], const double bc_re[4], const double bc_im[4], double kappa, int eo) {
    fields_t f;
    if (!out || setup(&f, U, u_f32, psi, psi_f32, dims, bc_re, bc_im)) return 1;
    const size_t n = (size_t)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    if (eo == 0) {
        hop_field(out, &f, -1);
        for (size_t k = 0; k < n; ++k) out[k] = ld(psi, k, psi_f32) - kappa * out[k];
        return 0;
    }
    if (eo != 1) return 1;
    for (int mu = 0; mu < 4; ++mu)
        if (dims[mu] & 1) return 1;
    cplx *tmp = (cplx *)malloc(n * sizeof(cplx));
    if (!tmp) return 2;
    hop_field(tmp, &f, 1); /* tmp_o = H_oe psi_e */
    fields_t g = f;
    g.psi = tmp;
    g.psi_f32 = 0;
    hop_field(out, &g, 0); /* out_e = H_eo tmp_o */
    const int X = dims[0], Y = dims[1], Z = dims[2];
    for (size_t site = 0; site < n / 12; ++site) {
        size_t r = site;
        int x0 = (int)(r % X); r /= X;
        int x1 = (int)(r % Y); r /= Y;
        int x2 = (int)(r % Z); r /= Z;
        int x3 = (int)r;
        int even = ((x0 + x1 + x2 + x3) & 1) == 0;
        for (int k = 0; k < 12; ++k) {
            size_t idx = site * 12 + k;
            out[idx] = even ? ld(psi, idx, psi_f32) - kappa * kappa * out[idx] : 0;
        }
    }
    free(tmp);
    return 0;
}

/* ---- next row f1: twisted-mass Wilson fermions ("N_f = 2 twisted-mass Wilson fermions [18, 21]",
 * "even-odd preconditioning"; the paper prints no formula -- DESIGN.md reading F1) -------------------------
 *   M_tm(mu)     = (1 + 2 i kappa mu gamma_5) - kappa H                         (one flavour; the other has -mu)
 *   Mhat_tm(mu)  = (1 + 2 i kappa mu gamma_5) - kappa^2 H_eo (1 + 2 i kappa mu gamma_5)^-1 H_oe   on even sites
 * i.e. the Schur complement of M_tm with respect to the odd sites.  The site-diagonal matrix and its inverse
 * are built as dense 4x4 complex matrices; the inverse by Gauss-Jordan elimination, not by the closed form. */
static void tm_diag(cplx d[4][4], double theta) {
    for (int s = 0; s < 4; ++s)
        for (int t = 0; t < 4; ++t) d[s][t] = (s == t ? 1.0 : 0.0) + I * theta * GAMMA[4][s][t];
}

static int inv4(cplx inv[4][4], cplx a[4][4]) {
    cplx m[4][8];
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 8; ++c) m[r][c] = c < 4 ? a[r][c] : (c - 4 == r ? 1.0 : 0.0);
    for (int col = 0; col < 4; ++col) {
        int piv = col;
        for (int r = col + 1; r < 4; ++r)
            if (cabs(m[r][col]) > cabs(m[piv][col])) piv = r;
        if (cabs(m[piv][col]) == 0.0) return 1;
        for (int c = 0; c < 8; ++c) { cplx t = m[col][c]; m[col][c] = m[piv][c]; m[piv][c] = t; }
        cplx d = m[col][col];
        for (int c = 0; c < 8; ++c) m[col][c] /= d;
        for (int r = 0; r < 4; ++r)
            if (r != col) {
                cplx fct = m[r][col];
                for (int c = 0; c < 8; ++c) m[r][c] -= fct * m[col][c];
            }
    }
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 4; ++c) inv[r][c] = m[r][c + 4];
    return 0;
}

/* v <- d v for every site of the field (12 complex per site, spin-major) */
static void spin_mul_field(cplx *v, size_t nsites, cplx d[4][4]) {
#pragma omp parallel for schedule(static)
    for (long n = 0; n < (long)nsites; ++n) {
        cplx t[4][3];
        for (int s = 0; s < 4; ++s)
            for (int a = 0; a < 3; ++a) {
                cplx acc = 0;
                for (int sp = 0; sp < 4; ++sp) acc += d[s][sp] * v[(size_t)n * 12 + sp * 3 + a];
                t[s][a] = acc;
            }
        for (int s = 0; s < 4; ++s)
            for (int a = 0; a < 3; ++a) v[(size_t)n * 12 + s * 3 + a] = t[s][a];
    }
}

/* eo = 0: out = (1 + 2 i kappa mu g5) psi - kappa H psi on all sites.
 * eo = 1: out_e = (1 + 2 i kappa mu g5) psi_e - kappa^2 H_eo (1 + 2 i kappa mu g5)^-1 H_oe psi_e, zero on odd sites. */
int oracle_apply_M_tm(double complex *out, const void *U, int u_f32, const void *psi, int psi_f32,
                      const int dims[4], const double bc_re[4], const double bc_im[4], double kappa, double mu,
                      int eo) {
    fields_t f;
    if (!out || setup(&f, U, u_f32, psi, psi_f32, dims, bc_re, bc_im)) return 1;
    if (eo != 0 && eo != 1) return 1;
    const size_t nsites = (size_t)dims[0] * dims[1] * dims[2] * dims[3], n = nsites * 12;
    cplx d[4][4], dinv[4][4];
    tm_diag(d, 2.0 * kappa * mu);
    if (inv4(dinv, d)) return 3;
    cplx *diag = (cplx *)malloc(n * sizeof(cplx)); /* (1 + 2 i kappa mu g5) psi */
    if (!diag) return 2;
    for (size_t k = 0; k < n; ++k) diag[k] = ld(psi, k, psi_f32);
    spin_mul_field(diag, nsites, d);
    if (eo == 0) {
        hop_field(out, &f, -1);
        for (size_t k = 0; k < n; ++k) out[k] = diag[k] - kappa * out[k];
        free(diag);
        return 0;
    }
    for (int m = 0; m < 4; ++m)
        if (dims[m] & 1) { free(diag); return 1; }
    cplx *tmp = (cplx *)malloc(n * sizeof(cplx));
    if (!tmp) { free(diag); return 2; }
    hop_field(tmp, &f, 1);               /* tmp_o = H_oe psi_e */
    spin_mul_field(tmp, nsites, dinv);   /* tmp_o = (1 + 2 i kappa mu g5)^-1 tmp_o  (zero stays zero on even sites) */
    fields_t g = f;
    g.psi = tmp;
    g.psi_f32 = 0;
    hop_field(out, &g, 0);               /* out_e = H_eo tmp_o */
    const int X = dims[0], Y = dims[1], Z = dims[2];
    for (size_t site = 0; site < nsites; ++site) {
        size_t r = site;
        int x0 = (int)(r % X); r /= X;
        int x1 = (int)(r % Y); r /= Y;
        int x2 = (int)(r % Z); r /= Z;
        int x3 = (int)r;
        int even = ((x0 + x1 + x2 + x3) & 1) == 0;
        for (int k = 0; k < 12; ++k) {
            size_t idx = site * 12 + k;
            out[idx] = even ? diag[idx] - kappa * kappa * out[idx] : 0;
        }
    }
    free(tmp);
    free(diag);
    return 0;
}

/* (H psi)(x) at n listed sites; coords [n][4] = (x,y,z,t); out [n][4][3].  For sampled parity at full size. */
int oracle_dslash_sites(double complex *out, const void *U, int u_f32, const void *psi, int psi_f32,
                        const int dims[4], const double bc_re[4], const double bc_im[4], const int *coords,
                        long n) {
    fields_t f;
    if (!out || !coords || setup(&f, U, u_f32, psi, psi_f32, dims, bc_re, bc_im)) return 1;
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) hop_site((cplx(*)[3])(out + k * 12), &f, coords + 4 * k, NULL);
    return 0;
}

/* (M psi)(x) at n listed sites.  eo = 0: psi(x) - kappa (H psi)(x).
 * eo = 1: psi(x) - kappa^2 (H H psi)(x); on an even x this is M_eo, because H maps even->odd->even. */
int oracle_apply_M_sites(double complex *out, const void *U, int u_f32, const void *psi, int psi_f32,
                         const int dims[4], const double bc_re[4], const double bc_im[4], double kappa,
                         int eo, const int *coords, long n) {
    fields_t f;
    if (!out || !coords || setup(&f, U, u_f32, psi, psi_f32, dims, bc_re, bc_im)) return 1;
    if (eo != 0 && eo != 1) return 1;
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) {
        const int *x = coords + 4 * k;
        cplx acc[4][3];
        if (eo == 0) {
            hop_site(acc, &f, x, NULL);
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) out[k * 12 + s * 3 + a] = spinor(&f, x, s, a) - kappa * acc[s][a];
        } else {
            cplx nb[8][4][3];
            for (int mu = 0; mu < 4; ++mu) {
                int y[4] = {x[0], x[1], x[2], x[3]};
                y[mu] = (x[mu] + 1 + f.L[mu]) % f.L[mu];
                hop_site(nb[2 * mu], &f, y, NULL);
                y[mu] = (x[mu] - 1 + f.L[mu]) % f.L[mu];
                hop_site(nb[2 * mu + 1], &f, y, NULL);
            }
            hop_site(acc, &f, x, nb);
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a)
                    out[k * 12 + s * 3 + a] = spinor(&f, x, s, a) - kappa * kappa * acc[s][a];
        }
    }
    return 0;
}

/* Appendix A.7: third row of an SU(3) matrix from the first two, row2 = conj(row0 x row1). */
void oracle_recon_row2(const double complex *r0, const double complex *r1, double complex *r2) {
    r2[0] = conj(r0[1] * r1[2] - r0[2] * r1[1]);
    r2[1] = conj(r0[2] * r1[0] - r0[0] * r1[2]);
    r2[2] = conj(r0[0] * r1[1] - r0[1] * r1[0]);
}
