/* hisq_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, definition-level fp64 implementation of what the hot path computes: the HISQ
 * staggered Dslash of arXiv:2306.01098 (Sec. 5.1), its even/odd restrictions
 * D_eo / D_oe, the normal operator A = m^2 - D_eo D_oe (PAPER.md:139-141 `applyMdaggM`, with
 * M = Dslash + m from Eq. (1)) and a textbook conjugate gradient on it.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code, header, table or constant with paper_2306_01098_b200/csrc.
 *
 * Storage is deliberately unlike the GPU's: everything lives on the FULL lattice in lexicographic
 * order, lex = x + Lx*(y + Ly*(z + Lz*t)), parity is handled by masking:
 *      links  F[lex][mu][a][b]   (9 complex, row major, (U phi)_a = sum_b U_ab phi_b)
 *      field  phi[k][lex][c]     (k = right-hand side, c = colour)
 * mu = 0,1,2,3 <-> x,y,z,t.  All coefficients and staggered phases are already
 * folded into the link arrays by whoever generated them ("we ignore constants and
 * the staggered phases"; readings R6/R7).
 *
 * The operator (with the two misprints read as DESIGN.md R1/R2: mu runs over the
 * four directions, and the forward Naik link is W_{x,mu}):
 *
 *   (D phi)(x) = sum_mu [ ( X_mu(x) phi(x+mu) - X_mu(x-mu)^+ phi(x-mu) )
 *                       + ( W_mu(x) phi(x+3mu) - W_mu(x-3mu)^+ phi(x-3mu) ) ]
 *
 * Coordinates are periodic (gauge field periodic); the spinor field is periodic in
 * space and ANTI-periodic in time: a gathered phi picks up -1 exactly when its
 * t-hop leaves [0, Lt).
 *
 * Arithmetic order follows the paper's operation count: per direction four complex
 * 3x3 mat-vecs (66 flop each) and three vector additions; then three more vector additions to
 * combine the four directions: 4*(4*66 + 3*6) + 3*6 = 1146.  Build with -DORACLE_COUNT to make the
 * helpers count flops and words so that tests can check 1146 / 288 / 96 / 6 (pin P1).
 *
 * Pins (tests/test_oracle_pins.py): P1 counts, P2 free-field closed form, P3 anti-Hermiticity,
 * P4 gauge covariance, P5 parity, P6 boundary-sign folding, P7 dense 4^4 brute force, P8 point
 * source, P9 linearity, P10 index bijection, P11/P12 CG, P15 full-matrix solve (dense M on 4^4).
 * Parity UNPINNED: nothing here.
 */
#include <complex.h>
#ifdef _OPENMP
#include <omp.h>
#endif
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#ifdef ORACLE_COUNT
static long long cnt_flop, cnt_link_words, cnt_vec_words, cnt_out_words;
#define COUNT_FLOP(n) (cnt_flop += (n))
#define COUNT_LINK(n) (cnt_link_words += (n))
#define COUNT_VEC(n) (cnt_vec_words += (n))
#define COUNT_OUT(n) (cnt_out_words += (n))
void oracle_count_reset(void) { cnt_flop = cnt_link_words = cnt_vec_words = cnt_out_words = 0; }
void oracle_count_get(long long *c) { c[0] = cnt_flop; c[1] = cnt_link_words; c[2] = cnt_vec_words; c[3] = cnt_out_words; }
#else
#define COUNT_FLOP(n)
#define COUNT_LINK(n)
#define COUNT_VEC(n)
#define COUNT_OUT(n)
#endif

/* ---------- coordinates ---------- */

static long lex_of(const int *L, const int *c)
{
    return c[0] + (long)L[0] * (c[1] + (long)L[1] * (c[2] + (long)L[2] * c[3]));
}

static void coords_of(const int *L, long lex, int *c)
{
    c[0] = (int)(lex % L[0]); lex /= L[0];
    c[1] = (int)(lex % L[1]); lex /= L[1];
    c[2] = (int)(lex % L[2]); lex /= L[2];
    c[3] = (int)lex;
}

static long volume_of(const int *L) { return (long)L[0] * L[1] * L[2] * L[3]; }

/* Eq. (4) PAPER.md:447-454 read with integer floor (R3):
 *   index = floor(lex/2) + (V/2) * ((x+y+z+t) mod 2)                                  */
void oracle_eo_index(const int *L, long *eo)
{
    long V = volume_of(L);
    for (long lex = 0; lex < V; ++lex) {
        int c[4];
        coords_of(L, lex, c);
        eo[lex] = lex / 2 + (V / 2) * ((c[0] + c[1] + c[2] + c[3]) % 2);
    }
}

/* Eq. (5): link (x, mu) at  eo(x) + mu*V. */
void oracle_link_index(const int *L, long *slot /* [V][4] */)
{
    long V = volume_of(L);
    for (long lex = 0; lex < V; ++lex) {
        int c[4];
        coords_of(L, lex, c);
        long eo = lex / 2 + (V / 2) * ((c[0] + c[1] + c[2] + c[3]) % 2);
        for (int mu = 0; mu < 4; ++mu) slot[lex * 4 + mu] = eo + (long)mu * V;
    }
}

/* ---------- the four helpers the flop count is made of ---------- */

/* r = U v : 9 complex multiplies (6 flop) + 6 complex adds (2 flop) = 66 flop */
static void mat_vec(const cplx *U, const cplx *v, cplx *r)
{
    for (int a = 0; a < 3; ++a)
        r[a] = (U[3 * a + 0] * v[0] + U[3 * a + 1] * v[1]) + U[3 * a + 2] * v[2];
    COUNT_FLOP(66); COUNT_LINK(18); COUNT_VEC(6);
}

/* r = U^dagger v : (U^+)_ab = conj(U_ba); same 66 flop (conjugation is a sign, not counted) */
static void matdag_vec(const cplx *U, const cplx *v, cplx *r)
{
    for (int a = 0; a < 3; ++a)
        r[a] = (conj(U[0 + a]) * v[0] + conj(U[3 + a]) * v[1]) + conj(U[6 + a]) * v[2];
    COUNT_FLOP(66); COUNT_LINK(18); COUNT_VEC(6);
}

static void vec_add(const cplx *a, const cplx *b, cplx *r)
{
    for (int c = 0; c < 3; ++c) r[c] = a[c] + b[c];
    COUNT_FLOP(6);
}

static void vec_sub(const cplx *a, const cplx *b, cplx *r)
{
    for (int c = 0; c < 3; ++c) r[c] = a[c] - b[c];
    COUNT_FLOP(6);
}

/* phi(y) as seen from a hop: times -1 if the hop crossed the t boundary. */
static void gather(const cplx *phi, long y, int sign, cplx *v)
{
    for (int c = 0; c < 3; ++c) v[c] = (sign < 0) ? -phi[3 * y + c] : phi[3 * y + c];
}

/* ---------- D on one site ---------- */

static void dslash_site(const int *L, const cplx *X, const cplx *W, const cplx *phi, long lex, cplx *out)
{
    int x[4];
    coords_of(L, lex, x);
    cplx dir[4][3];
    for (int mu = 0; mu < 4; ++mu) {
        cplx term[2][3];
        for (int f = 0; f < 2; ++f) {
            const cplx *F = f ? W : X;
            int hop = f ? 3 : 1;
            int yp[4] = { x[0], x[1], x[2], x[3] }, ym[4] = { x[0], x[1], x[2], x[3] };
            yp[mu] = (x[mu] + hop) % L[mu];
            ym[mu] = ((x[mu] - hop) % L[mu] + L[mu]) % L[mu];
            int sp = (mu == 3 && x[3] + hop >= L[3]) ? -1 : +1;
            int sm = (mu == 3 && x[3] - hop < 0) ? -1 : +1;
            long lp = lex_of(L, yp), lm = lex_of(L, ym);
            cplx vp[3], vm[3], fwd[3], bwd[3];
            gather(phi, lp, sp, vp);
            gather(phi, lm, sm, vm);
            mat_vec(F + (lex * 4 + mu) * 9, vp, fwd);     /* F_mu(x)        phi(x + hop mu) */
            matdag_vec(F + (lm * 4 + mu) * 9, vm, bwd);   /* F_mu(x-hop mu)^+ phi(x - hop mu) */
            vec_sub(fwd, bwd, term[f]);
        }
        vec_add(term[0], term[1], dir[mu]);
    }
    cplx s01[3], s012[3];
    vec_add(dir[0], dir[1], s01);
    vec_add(s01, dir[2], s012);
    vec_add(s012, dir[3], out);
    COUNT_OUT(6);
}

/* The same sum for ONE site whose 16 links and 16 neighbour vectors were fetched by the caller (used to
 * check sampled outputs of lattices too big to hold on the host): Ff[f][mu] = F_mu(x), Fb[f][mu] =
 * F_mu(x - hop mu), vp[f][mu] = phi(x + hop mu), vm[f][mu] = phi(x - hop mu), f = 0 fat (hop 1), 1 Naik
 * (hop 3); t, Lt give the antiperiodic sign.  Same helpers, same order as dslash_site. */
static void dslash_site_gathered(int t, int Lt, const cplx *Ff, const cplx *Fb, const cplx *vp_in, const cplx *vm_in,
                                 cplx *out)
{
    cplx dir[4][3];
    for (int mu = 0; mu < 4; ++mu) {
        cplx term[2][3];
        for (int f = 0; f < 2; ++f) {
            int hop = f ? 3 : 1;
            int sp = (mu == 3 && t + hop >= Lt) ? -1 : +1;
            int sm = (mu == 3 && t - hop < 0) ? -1 : +1;
            cplx vp[3], vm[3], fwd[3], bwd[3];
            gather(vp_in + (f * 4 + mu) * 3, 0, sp, vp);
            gather(vm_in + (f * 4 + mu) * 3, 0, sm, vm);
            mat_vec(Ff + (f * 4 + mu) * 9, vp, fwd);
            matdag_vec(Fb + (f * 4 + mu) * 9, vm, bwd);
            vec_sub(fwd, bwd, term[f]);
        }
        vec_add(term[0], term[1], dir[mu]);
    }
    cplx s01[3], s012[3];
    vec_add(dir[0], dir[1], s01);
    vec_add(s01, dir[2], s012);
    vec_add(s012, dir[3], out);
}

/* n sites: t[i]; Ff, Fb [i][2][4][9]; vp, vm [i][2][4][3]; out [i][3]. */
void oracle_dslash_gathered(int Lt, long n, const int *t, const cplx *Ff, const cplx *Fb, const cplx *vp, const cplx *vm,
                            cplx *out)
{
    for (long i = 0; i < n; ++i)
        dslash_site_gathered(t[i], Lt, Ff + i * 72, Fb + i * 72, vp + i * 24, vm + i * 24, out + i * 3);
}

/* ---------- D on sets of sites ---------- */

static int parity_of(const int *L, long lex)
{
    int c[4];
    coords_of(L, lex, c);
    return (c[0] + c[1] + c[2] + c[3]) & 1;
}

/* out(x) = (D phi)(x) for every site whose parity is in `rows` (bit 0: even rows, bit 1: odd
 * rows; 3 = the full-lattice D); other rows of `out` are set to zero. */
void oracle_dslash_rows(const int *L, const cplx *X, const cplx *W, const cplx *phi, cplx *out,
                        int nrhs, int rows)
{
    long V = volume_of(L);
    for (int k = 0; k < nrhs; ++k) {
        const cplx *p = phi + (long)k * V * 3;
        cplx *o = out + (long)k * V * 3;
#ifndef ORACLE_COUNT
#pragma omp parallel for schedule(static)
#endif
        for (long lex = 0; lex < V; ++lex) {
            if ((rows >> parity_of(L, lex)) & 1)
                dslash_site(L, X, W, p, lex, o + 3 * lex);
            else
                o[3 * lex] = o[3 * lex + 1] = o[3 * lex + 2] = 0.0;
        }
    }
}

/* (D phi)(x) at a list of sites only (sampled parity checks on big lattices). out[k][i][c]. */
void oracle_dslash_at(const int *L, const cplx *X, const cplx *W, const cplx *phi, cplx *out,
                      int nrhs, const long *sites, long nsites)
{
    long V = volume_of(L);
    for (int k = 0; k < nrhs; ++k) {
#ifndef ORACLE_COUNT
#pragma omp parallel for schedule(static)
#endif
        for (long i = 0; i < nsites; ++i)
            dslash_site(L, X, W, phi + (long)k * V * 3, sites[i], out + ((long)k * nsites + i) * 3);
    }
}

/* D_eo / D_oe (north_star): `parity` is the parity of the OUTPUT sites.
 * Zero phi on the output parity, apply D, keep the output parity. */
void oracle_dslash_parity(const int *L, const cplx *X, const cplx *W, const cplx *phi, cplx *out,
                          int nrhs, int parity)
{
    long V = volume_of(L);
    cplx *masked = (cplx *)malloc(sizeof(cplx) * 3 * V * nrhs);
    for (int k = 0; k < nrhs; ++k)
        for (long lex = 0; lex < V; ++lex) {
            int keep = parity_of(L, lex) != parity;
            for (int c = 0; c < 3; ++c) {
                long i = ((long)k * V + lex) * 3 + c;
                masked[i] = keep ? phi[i] : 0.0;
            }
        }
    oracle_dslash_rows(L, X, W, masked, out, nrhs, 1 << parity);
    free(masked);
}

/* A v = m^2 v - D_eo D_oe v on even sites (M = D + m, Eq. (1), and
 * D^+ = -D give M^+ M = m^2 - D^2, whose even-even block is m^2 - D_eo D_oe).  v and out are
 * full-lattice fields; odd sites of v are ignored, odd sites of out are zero. */
void oracle_apply_A(const int *L, const cplx *X, const cplx *W, double mass, const cplx *v, cplx *out,
                    int nrhs)
{
    long V = volume_of(L);
    long n = 3 * V * nrhs;
    cplx *t_o = (cplx *)malloc(sizeof(cplx) * n);
    oracle_dslash_parity(L, X, W, v, t_o, nrhs, 1);   /* t_o = D_oe v_e */
    oracle_dslash_parity(L, X, W, t_o, out, nrhs, 0); /* out = D_eo t_o */
    for (int k = 0; k < nrhs; ++k)
        for (long lex = 0; lex < V; ++lex) {
            int even = parity_of(L, lex) == 0;
            for (int c = 0; c < 3; ++c) {
                long i = ((long)k * V + lex) * 3 + c;
                out[i] = even ? mass * mass * v[i] - out[i] : 0.0;
            }
        }
    free(t_o);
}

/* ---------- textbook CG (Hestenes-Stiefel), one right-hand side at a time ---------- */

static double re_dot(const cplx *a, const cplx *b, long n)
{
    double s = 0.0;
    for (long i = 0; i < n; ++i) s += creal(conj(a[i]) * b[i]);
    return s;
}

/* Solve A x_k = b_k for k < nrhs, x_0 = 0; stop when ||r|| <= tol ||b|| (norm, not squared;
 * DESIGN.md R10).  Only even sites of b are used.  iters[k] = iterations taken,
 * relres[k] = ||b - A x|| / ||b|| recomputed at the end.  Returns 0, or 1 if some RHS hit max_iter.
 * If resid_hist != NULL it receives sqrt(rho_i)/||b|| for RHS 0, i = 0..min(iters, hist_len-1). */
int oracle_cg(const int *L, const cplx *X, const cplx *W, double mass, double tol, int max_iter,
              const cplx *b, cplx *x, int nrhs, int *iters, double *relres,
              double *resid_hist, int hist_len)
{
    long V = volume_of(L);
    long n = 3 * V;
    int status = 0;
    cplx *r = (cplx *)malloc(sizeof(cplx) * n), *p = (cplx *)malloc(sizeof(cplx) * n),
         *q = (cplx *)malloc(sizeof(cplx) * n), *bk = (cplx *)malloc(sizeof(cplx) * n);
    for (int k = 0; k < nrhs; ++k) {
        cplx *xk = x + (long)k * n;
        for (long lex = 0; lex < V; ++lex)
            for (int c = 0; c < 3; ++c)
                bk[3 * lex + c] = parity_of(L, lex) == 0 ? b[(long)k * n + 3 * lex + c] : 0.0;
        memset(xk, 0, sizeof(cplx) * n);
        memcpy(r, bk, sizeof(cplx) * n);
        memcpy(p, bk, sizeof(cplx) * n);
        double bb = re_dot(bk, bk, n), rho = bb;
        int it = 0;
        if (resid_hist && k == 0 && hist_len > 0) resid_hist[0] = 1.0;
        while (bb > 0.0 && sqrt(rho) > tol * sqrt(bb)) {
            if (it >= max_iter) { status = 1; break; }
            oracle_apply_A(L, X, W, mass, p, q, 1);
            double alpha = rho / re_dot(p, q, n);
            for (long i = 0; i < n; ++i) xk[i] += alpha * p[i];
            for (long i = 0; i < n; ++i) r[i] -= alpha * q[i];
            double rho_new = re_dot(r, r, n);
            ++it;
            if (resid_hist && k == 0 && it < hist_len) resid_hist[it] = sqrt(rho_new / bb);
            double beta = rho_new / rho;
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
            rho = rho_new;
        }
        iters[k] = it;
        oracle_apply_A(L, X, W, mass, xk, q, 1);
        for (long i = 0; i < n; ++i) q[i] = bk[i] - q[i];
        relres[k] = bb > 0.0 ? sqrt(re_dot(q, q, n) / bb) : 0.0;
    }
    free(r); free(p); free(q); free(bk);
    return status;
}

/* ---------- the full fermion matrix M = D + m (Eq. (1) PAPER.md:131 writes det(D + m)) ---------- */

/* out = (D + m) phi on the whole lattice (both parities). */
void oracle_apply_M(const int *L, const cplx *X, const cplx *W, double mass, const cplx *phi, cplx *out,
                    int nrhs)
{
    long n = 3 * volume_of(L) * nrhs;
    oracle_dslash_rows(L, X, W, phi, out, nrhs, 3);
    for (long i = 0; i < n; ++i) out[i] += mass * phi[i];
}

/* Solve M x_k = b_k on the WHOLE lattice, x_0 = 0, by textbook CG on the normal equations
 *      M^+ M x = M^+ b,   M^+ = m - D  (D^+ = -D, pin P3),   M^+ M = m^2 - D D
 * written with full-lattice operators only -- no even-odd decomposition, no Schur complement: this is the
 * plain definition the GPU's even-odd preconditioned solve must reproduce.
 * Stop when ||M^+ b - M^+ M x|| <= tol ||M^+ b||; relres[k] = ||b - M x|| / ||b|| recomputed at the end
 * (the quantity the GPU call bounds).  Returns 0, or 1 if some RHS hit max_iter. */
int oracle_solve_M(const int *L, const cplx *X, const cplx *W, double mass, double tol, int max_iter,
                   const cplx *b, cplx *x, int nrhs, int *iters, double *relres)
{
    long V = volume_of(L);
    long n = 3 * V;
    int status = 0;
    cplx *r = (cplx *)malloc(sizeof(cplx) * n), *p = (cplx *)malloc(sizeof(cplx) * n),
         *q = (cplx *)malloc(sizeof(cplx) * n), *t = (cplx *)malloc(sizeof(cplx) * n);
    for (int k = 0; k < nrhs; ++k) {
        const cplx *bk = b + (long)k * n;
        cplx *xk = x + (long)k * n;
        memset(xk, 0, sizeof(cplx) * n);
        /* r = M^+ b = m b - D b */
        oracle_dslash_rows(L, X, W, bk, t, 1, 3);
        for (long i = 0; i < n; ++i) r[i] = mass * bk[i] - t[i];
        memcpy(p, r, sizeof(cplx) * n);
        double cc = re_dot(r, r, n), rho = cc;
        int it = 0;
        while (cc > 0.0 && sqrt(rho) > tol * sqrt(cc)) {
            if (it >= max_iter) { status = 1; break; }
            /* q = M^+ M p = m^2 p - D (D p) */
            oracle_dslash_rows(L, X, W, p, t, 1, 3);
            oracle_dslash_rows(L, X, W, t, q, 1, 3);
            for (long i = 0; i < n; ++i) q[i] = mass * mass * p[i] - q[i];
            double alpha = rho / re_dot(p, q, n);
            for (long i = 0; i < n; ++i) xk[i] += alpha * p[i];
            for (long i = 0; i < n; ++i) r[i] -= alpha * q[i];
            double rho_new = re_dot(r, r, n);
            ++it;
            double beta = rho_new / rho;
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
            rho = rho_new;
        }
        iters[k] = it;
        oracle_apply_M(L, X, W, mass, xk, q, 1);
        for (long i = 0; i < n; ++i) q[i] = bk[i] - q[i];
        double bb = re_dot(bk, bk, n);
        relres[k] = bb > 0.0 ? sqrt(re_dot(q, q, n) / bb) : 0.0;
    }
    free(r); free(p); free(q); free(t);
    return status;
}

int oracle_threads(void)
{
    int n = 1;
#if defined(_OPENMP) && !defined(ORACLE_COUNT)
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
