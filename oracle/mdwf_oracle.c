/* ORACLE-B (test infrastructure only) -- plain C restatement of arXiv 2104.05615.
 *
 * Plain site loops in double precision, no blocking, no fusion, no intrinsics; OpenMP
 * "parallel for" over sites is the only concession to speed.  Shares NO code, header, table
 * or constant generator with the CUDA path in paper_2104_05615_b200/csrc.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liboracle.so mdwf_oracle.c -lm   (see oracle/build.py)
 *
 * Citations are to /root/reference/PAPER.md lines; R1..R20 are the readings listed in DESIGN.md.
 *
 * Field layout inside the oracle: a "box" is a 4D array of sites (x fastest) with per-direction
 * periodic / open flags and a global origin.  f[s][site][spin][colour] double complex, BOTH
 * parities stored.  The whole lattice is the box with every direction periodic.
 *
 * Pinned by tests/test_oracle_*.py: free-field momentum-space closed form, Shamir limit,
 * gamma5-hermiticity, Schur identity, gauge covariance, dense direct solves, and agreement with
 * the independent numpy restatement oracle/mdwf.py to <= 1e-13.
 */
#include <complex.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

typedef struct {
  int n[4];    /* extents x,y,z,t */
  int per[4];  /* 1 = periodic wrap, 0 = zero Dirichlet at the array edge */
  int org[4];  /* global coordinate of local (0,0,0,0) */
  long V;      /* sites */
} box_t;

typedef struct {
  int L[4], Ls, B[4];
  double b, c, M5, mf, alpha, beta;
  long V4;
  cplx *U;           /* [mu][lex][3][3], t-boundary sign folded in (R7) */
  double *m5p, *mphip, *m5invp; /* P+ blocks, Ls x Ls, row major (R3, R4) */
  cplx gam[4][4][4]; /* R2 */
  box_t lat, blk;
  int nblk, nb[4];
  long n_inner_applies;
} ora_t;

/* ---- R2: gamma matrices, chiral basis, gamma5 = diag(1,1,-1,-1) ------------------------------ */
static void set_gamma(ora_t *o) {
  static const cplx sig[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I}, {I, 0}}, {{1, 0}, {0, -1}}};
  memset(o->gam, 0, sizeof(o->gam));
  for (int k = 0; k < 3; k++)
    for (int a = 0; a < 2; a++)
      for (int b2 = 0; b2 < 2; b2++) {
        o->gam[k][a][2 + b2] = -I * sig[k][a][b2];
        o->gam[k][2 + a][b2] = I * sig[k][a][b2];
      }
  for (int a = 0; a < 2; a++) { o->gam[3][a][2 + a] = 1; o->gam[3][2 + a][a] = 1; }
}

/* ---- R3/R4: Ls x Ls chirality blocks --------------------------------------------------------- */
static void set_5d(ora_t *o) {
  int Ls = o->Ls;
  o->alpha = o->b * (4.0 - o->M5) + 1.0;  /* PAPER.md:91 eq. 4 diagonal blocks, R1 */
  o->beta = o->c * (4.0 - o->M5) - 1.0;
  o->m5p = calloc(Ls * Ls, sizeof(double));
  o->mphip = calloc(Ls * Ls, sizeof(double));
  o->m5invp = calloc(Ls * Ls, sizeof(double));
  for (int s = 0; s < Ls; s++) {
    /* S_minus: (S psi)_s = psi_{s-1}, (S psi)_0 = -mf psi_{Ls-1} */
    int sm = (s + Ls - 1) % Ls;
    double w = (s == 0) ? -o->mf : 1.0;
    o->m5p[s * Ls + s] += o->alpha;
    o->m5p[s * Ls + sm] += o->beta * w;
    o->mphip[s * Ls + s] += -0.5 * o->b;   /* PAPER.md:101 eq. 7, R1: Mphi = -(b + c L)/2 */
    o->mphip[s * Ls + sm] += -0.5 * o->c * w;
  }
  double k = o->beta / o->alpha;
  double den = o->alpha * (1.0 + o->mf * pow(-k, Ls));
  for (int s = 0; s < Ls; s++)
    for (int sp = 0; sp < Ls; sp++)
      o->m5invp[s * Ls + sp] = pow(-k, (s - sp + Ls) % Ls) * (s >= sp ? 1.0 : -o->mf) / den; /* R4 */
}

static void box_init(box_t *bx, const int n[4], const int per[4], const int org[4]) {
  bx->V = 1;
  for (int d = 0; d < 4; d++) { bx->n[d] = n[d]; bx->per[d] = per[d]; bx->org[d] = org[d]; bx->V *= n[d]; }
}

static inline void lex2c(const box_t *bx, long i, int c[4]) {
  for (int d = 0; d < 4; d++) { c[d] = (int)(i % bx->n[d]); i /= bx->n[d]; }
}
static inline long c2lex(const int n[4], const int c[4]) {
  return c[0] + (long)n[0] * (c[1] + (long)n[1] * (c[2] + (long)n[2] * c[3]));
}
static inline long glob_site(const ora_t *o, const box_t *bx, const int c[4]) {
  int g[4];
  for (int d = 0; d < 4; d++) { g[d] = (bx->org[d] + c[d]) % o->L[d]; if (g[d] < 0) g[d] += o->L[d]; }
  return c2lex(o->L, g);
}

ora_t *ora_create(const int L[4], int Ls, double b, double c, double M5, double mf, const int B[4]) {
  for (int d = 0; d < 4; d++)
    if (L[d] < 2 || L[d] % 2 || B[d] < 2 || B[d] % 2 || L[d] % B[d]) return NULL;
  if (Ls < 2) return NULL;
  ora_t *o = calloc(1, sizeof(ora_t));
  o->Ls = Ls; o->b = b; o->c = c; o->M5 = M5; o->mf = mf;
  o->V4 = 1; o->nblk = 1;
  int per1[4] = {1, 1, 1, 1}, org0[4] = {0, 0, 0, 0};
  for (int d = 0; d < 4; d++) { o->L[d] = L[d]; o->B[d] = B[d]; o->V4 *= L[d]; o->nb[d] = L[d] / B[d]; o->nblk *= o->nb[d]; }
  if (b * (4.0 - M5) + 1.0 == 0.0) { free(o); return NULL; }
  set_gamma(o);
  set_5d(o);
  box_init(&o->lat, L, per1, org0);
  /* padded block box, R10 (PAD): pad 2 on both sides of each CUT direction */
  int n[4], per[4];
  for (int d = 0; d < 4; d++) { int cut = B[d] != L[d]; n[d] = cut ? B[d] + 4 : L[d]; per[d] = !cut; }
  box_init(&o->blk, n, per, org0);
  o->U = calloc((size_t)4 * o->V4 * 9, sizeof(cplx));
  return o;
}

void ora_destroy(ora_t *o) {
  if (!o) return;
  free(o->U); free(o->m5p); free(o->mphip); free(o->m5invp); free(o);
}

void ora_get_matrix(const ora_t *o, int which, double *out) {
  const double *m = which == 0 ? o->m5p : which == 1 ? o->mphip : o->m5invp;
  memcpy(out, m, sizeof(double) * o->Ls * o->Ls);
}
void ora_get_gamma(const ora_t *o, double *out /* [4][4][4][2] */) {
  for (int m = 0; m < 4; m++) for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) {
    out[((m * 4 + i) * 4 + j) * 2] = creal(o->gam[m][i][j]);
    out[((m * 4 + i) * 4 + j) * 2 + 1] = cimag(o->gam[m][i][j]);
  }
}
long ora_inner_applies(const ora_t *o) { return o->n_inner_applies; }
int ora_num_blocks(const ora_t *o) { return o->nblk; }

/* ---- ABI layouts (include/mspcg.h): x_cb = lex/2 within a parity, parity = (x+y+z+t)%2 (eq. 3) -- */
static inline int site_parity(const int c[4]) { return (c[0] + c[1] + c[2] + c[3]) & 1; }

void ora_load_gauge(ora_t *o, const double *U_abi, int t_boundary) {
  long Vh = o->V4 / 2;
  for (int mu = 0; mu < 4; mu++)
    for (long i = 0; i < o->V4; i++) {
      int c[4]; lex2c(&o->lat, i, c);
      int p = site_parity(c);
      const double *src = U_abi + ((((size_t)mu * 2 + p) * Vh + i / 2) * 9) * 2;
      double sgn = (mu == 3 && c[3] == o->L[3] - 1 && t_boundary == -1) ? -1.0 : 1.0; /* R7 */
      for (int k = 0; k < 9; k++) o->U[((size_t)mu * o->V4 + i) * 9 + k] = sgn * (src[2 * k] + I * src[2 * k + 1]);
    }
}

static void unpack_even(const ora_t *o, const double *abi, cplx *f) {
  long Vh = o->V4 / 2;
  memset(f, 0, sizeof(cplx) * o->Ls * o->V4 * 12);
  for (int s = 0; s < o->Ls; s++)
    for (long i = 0; i < o->V4; i++) {
      int c[4]; lex2c(&o->lat, i, c);
      if (site_parity(c)) continue;
      const double *src = abi + (((size_t)s * Vh + i / 2) * 12) * 2;
      cplx *dst = f + ((size_t)s * o->V4 + i) * 12;
      for (int k = 0; k < 12; k++) dst[k] = src[2 * k] + I * src[2 * k + 1];
    }
}
static void pack_even(const ora_t *o, const cplx *f, double *abi) {
  long Vh = o->V4 / 2;
  for (int s = 0; s < o->Ls; s++)
    for (long i = 0; i < o->V4; i++) {
      int c[4]; lex2c(&o->lat, i, c);
      if (site_parity(c)) continue;
      double *dst = abi + (((size_t)s * Vh + i / 2) * 12) * 2;
      const cplx *src = f + ((size_t)s * o->V4 + i) * 12;
      for (int k = 0; k < 12; k++) { dst[2 * k] = creal(src[k]); dst[2 * k + 1] = cimag(src[k]); }
    }
}

/* ---- PAPER.md:105 eq. (8): D^w; dagger = gamma_mu -> -gamma_mu (R6) ---------------------------
 *   (D^w psi)(x) = sum_mu (1 - g_mu) U_mu(x) psi(x+mu) + (1 + g_mu) U_mu(x-mu)^dag psi(x-mu)
 * Links are read by GLOBAL periodic index (R10), neighbours outside an open box edge are zero. */
static void hop(const ora_t *o, const box_t *bx, const cplx *in, cplx *out, int dagger) {
  const double sg = dagger ? -1.0 : 1.0;
  const long V = bx->V;
#pragma omp parallel for schedule(static)
  for (long i = 0; i < V; i++) {
    int c[4]; lex2c(bx, i, c);
    long gx = glob_site(o, bx, c);
    for (int s = 0; s < o->Ls; s++) {
      cplx acc[4][3]; memset(acc, 0, sizeof(acc));
      for (int mu = 0; mu < 4; mu++) {
        for (int dir = 0; dir < 2; dir++) { /* 0: forward x+mu, 1: backward x-mu */
          int cn[4] = {c[0], c[1], c[2], c[3]};
          cn[mu] += dir == 0 ? 1 : -1;
          if (cn[mu] < 0 || cn[mu] >= bx->n[mu]) {
            if (!bx->per[mu]) continue;
            cn[mu] = (cn[mu] + bx->n[mu]) % bx->n[mu];
          }
          long j = c2lex(bx->n, cn);
          const cplx *psi = in + ((size_t)s * V + j) * 12;
          const cplx *u = o->U + ((size_t)mu * o->V4 + (dir == 0 ? gx : glob_site(o, bx, cn))) * 9;
          cplx h[4][3];
          for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) {
              cplx t = 0;
              for (int b2 = 0; b2 < 3; b2++)
                t += (dir == 0 ? u[a * 3 + b2] : conj(u[b2 * 3 + a])) * psi[sp * 3 + b2];
              h[sp][a] = t;
            }
          double gs = dir == 0 ? -sg : sg; /* (1 - g) forward, (1 + g) backward */
          for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) {
              cplx t = h[sp][a];
              for (int sq = 0; sq < 4; sq++) t += gs * o->gam[mu][sp][sq] * h[sq][a];
              acc[sp][a] += t;
            }
        }
      }
      memcpy(out + ((size_t)s * V + i) * 12, acc, sizeof(acc));
    }
  }
}

/* ---- 5D operators, diagonal in 4D; P+ block on spin 0,1 and its transpose on 2,3;
 *      dagger swaps them (R3).  Dense Ls x Ls product. ------------------------- */
static void apply5d(const ora_t *o, const box_t *bx, const double *mp, const cplx *in, cplx *out, int dagger) {
  const int Ls = o->Ls; const long V = bx->V;
#pragma omp parallel for schedule(static)
  for (long i = 0; i < V; i++)
    for (int s = 0; s < Ls; s++)
      for (int k = 0; k < 12; k++) {
        int upper = k < 6; /* spin 0,1 = P+ */
        int transpose = upper ? dagger : !dagger;
        cplx t = 0;
        for (int r = 0; r < Ls; r++)
          t += (transpose ? mp[r * Ls + s] : mp[s * Ls + r]) * in[((size_t)r * V + i) * 12 + k];
        out[((size_t)s * V + i) * 12 + k] = t;
      }
}

static void axpy(long n, double a, const cplx *x, cplx *y) {
#pragma omp parallel for schedule(static)
  for (long i = 0; i < n; i++) y[i] += a * x[i];
}
static void xmy(long n, const cplx *x, const cplx *y, cplx *out) { /* out = x - y */
#pragma omp parallel for schedule(static)
  for (long i = 0; i < n; i++) out[i] = x[i] - y[i];
}
static double rdot(long n, const cplx *x, const cplx *y) {
  double r = 0;
#pragma omp parallel for schedule(static) reduction(+ : r)
  for (long i = 0; i < n; i++) r += creal(x[i]) * creal(y[i]) + cimag(x[i]) * cimag(y[i]);
  return r;
}

/* ---- PAPER.md:95 eq. (5) and PAPER.md:232 eq. (15): D, D^dag, D^dag D factor by factor ----------- */
static void D_eo(const ora_t *o, const box_t *bx, const cplx *in, cplx *out, cplx *t1, cplx *t2, int dagger) {
  long n = (long)o->Ls * bx->V * 12;
  if (!dagger) {
    apply5d(o, bx, o->mphip, in, t1, 0);   /* Mphi           */
    hop(o, bx, t1, t2, 0);                 /* D^w  (M4oe)    */
    apply5d(o, bx, o->m5invp, t2, t1, 0);  /* M5^-1          */
    apply5d(o, bx, o->mphip, t1, t2, 0);   /* Mphi           */
    hop(o, bx, t2, t1, 0);                 /* D^w  (M4eo)    */
    apply5d(o, bx, o->m5invp, t1, t2, 0);  /* M5^-1          */
  } else {
    apply5d(o, bx, o->m5invp, in, t1, 1);  /* M5^-dag        */
    hop(o, bx, t1, t2, 1);                 /* D^w^dag        */
    apply5d(o, bx, o->mphip, t2, t1, 1);   /* Mphi^dag       */
    apply5d(o, bx, o->m5invp, t1, t2, 1);  /* M5^-dag        */
    hop(o, bx, t2, t1, 1);                 /* D^w^dag        */
    apply5d(o, bx, o->mphip, t1, t2, 1);   /* Mphi^dag       */
  }
  xmy(n, in, t2, out);                     /* 1 - (...)      */
}

typedef struct { cplx *t1, *t2, *t3; } tmp_t;
static tmp_t tmp_alloc(const ora_t *o, const box_t *bx) {
  size_t n = (size_t)o->Ls * bx->V * 12;
  tmp_t t = {calloc(n, sizeof(cplx)), calloc(n, sizeof(cplx)), calloc(n, sizeof(cplx))};
  return t;
}
static void tmp_free(tmp_t t) { free(t.t1); free(t.t2); free(t.t3); }

static void MdagM_box(const ora_t *o, const box_t *bx, const cplx *in, cplx *out, tmp_t w) {
  D_eo(o, bx, in, w.t3, w.t1, w.t2, 0);
  D_eo(o, bx, w.t3, out, w.t1, w.t2, 1);
}

/* ---- R10 (PAD): A_s = centre of (D^dag D on the zero-padded box) ------------------ */
static int in_centre(const ora_t *o, const box_t *bx, const int c[4]) {
  for (int d = 0; d < 4; d++)
    if (!bx->per[d] && (c[d] < 2 || c[d] >= 2 + o->B[d])) return 0;
  return 1;
}
static void zero_pad(const ora_t *o, const box_t *bx, cplx *f) {
  for (long i = 0; i < bx->V; i++) {
    int c[4]; lex2c(bx, i, c);
    if (in_centre(o, bx, c)) continue;
    for (int s = 0; s < o->Ls; s++) memset(f + ((size_t)s * bx->V + i) * 12, 0, 12 * sizeof(cplx));
  }
}
static void A_block(const ora_t *o, const box_t *bx, const cplx *in, cplx *out, tmp_t w) {
  MdagM_box(o, bx, in, out, w);
  zero_pad(o, bx, out);
}

static void block_box(const ora_t *o, int blk, box_t *bx) {
  *bx = o->blk;
  int r = blk;
  for (int d = 0; d < 4; d++) {
    int ob = (r % o->nb[d]) * o->B[d]; r /= o->nb[d];
    bx->org[d] = bx->per[d] ? 0 : ob - 2;
  }
}
/* copy block part of a lattice field into the centre of the box (pad = 0), or back */
static void box_gather(const ora_t *o, const box_t *bx, const cplx *lat, cplx *f, int scatter, cplx *lat_out) {
  for (long i = 0; i < bx->V; i++) {
    int c[4]; lex2c(bx, i, c);
    int cen = in_centre(o, bx, c);
    long g = glob_site(o, bx, c);
    for (int s = 0; s < o->Ls; s++) {
      cplx *b = f + ((size_t)s * bx->V + i) * 12;
      if (!scatter) {
        if (cen) memcpy(b, lat + ((size_t)s * o->V4 + g) * 12, 12 * sizeof(cplx));
        else memset(b, 0, 12 * sizeof(cplx));
      } else if (cen) {
        memcpy(lat_out + ((size_t)s * o->V4 + g) * 12, b, 12 * sizeof(cplx));
      }
    }
  }
}

/* ---- R13: k CG steps per block from a zero guess, own scalars per block ----- */
static void precond_lat(ora_t *o, const cplx *r_lat, cplx *z_lat, int k, int only_block) {
  box_t bx;
  size_t n = (size_t)o->Ls * o->blk.V * 12;
  cplx *x = malloc(n * sizeof(cplx)), *r = malloc(n * sizeof(cplx)), *p = malloc(n * sizeof(cplx)), *q = malloc(n * sizeof(cplx));
  tmp_t w = tmp_alloc(o, &o->blk);
  memset(z_lat, 0, sizeof(cplx) * o->Ls * o->V4 * 12);
  for (int blk = 0; blk < o->nblk; blk++) {
    if (only_block >= 0 && blk != only_block) continue;
    block_box(o, blk, &bx);
    box_gather(o, &bx, r_lat, r, 0, NULL);
    memset(x, 0, n * sizeof(cplx));
    memcpy(p, r, n * sizeof(cplx));
    double rho = rdot(n, r, r);
    for (int it = 0; it < k; it++) {
      if (rho == 0.0) break;
      A_block(o, &bx, p, q, w);
      o->n_inner_applies++;
      double pq = rdot(n, p, q);
      if (!(pq > 0.0)) break;
      double a = rho / pq;
      axpy(n, a, p, x);
      axpy(n, -a, q, r);
      double rho2 = rdot(n, r, r);
      double bt = rho2 / rho;
#pragma omp parallel for schedule(static)
      for (long i = 0; i < (long)n; i++) p[i] = r[i] + bt * p[i];
      rho = rho2;
    }
    box_gather(o, &bx, NULL, x, 1, z_lat);
  }
  free(x); free(r); free(p); free(q); tmp_free(w);
}

/* ---- ABI-level entry points -------------------------------------------------------------------- */
void ora_apply_D(ora_t *o, const double *in_abi, double *out_abi, int dagger) {
  size_t n = (size_t)o->Ls * o->V4 * 12;
  cplx *in = malloc(n * sizeof(cplx)), *out = malloc(n * sizeof(cplx));
  tmp_t w = tmp_alloc(o, &o->lat);
  unpack_even(o, in_abi, in);
  D_eo(o, &o->lat, in, out, w.t1, w.t2, dagger);
  pack_even(o, out, out_abi);
  free(in); free(out); tmp_free(w);
}

void ora_apply_MdagM(ora_t *o, const double *in_abi, double *out_abi) {
  size_t n = (size_t)o->Ls * o->V4 * 12;
  cplx *in = malloc(n * sizeof(cplx)), *out = malloc(n * sizeof(cplx));
  tmp_t w = tmp_alloc(o, &o->lat);
  unpack_even(o, in_abi, in);
  MdagM_box(o, &o->lat, in, out, w);
  pack_even(o, out, out_abi);
  free(in); free(out); tmp_free(w);
}

/* A_s applied to the block-`blk` part of an even lattice field; result on the block, zero elsewhere */
void ora_apply_A_block(ora_t *o, const double *in_abi, double *out_abi, int blk) {
  size_t n = (size_t)o->Ls * o->V4 * 12, nb = (size_t)o->Ls * o->blk.V * 12;
  cplx *in = malloc(n * sizeof(cplx)), *out = calloc(n, sizeof(cplx));
  cplx *bi = malloc(nb * sizeof(cplx)), *bo = malloc(nb * sizeof(cplx));
  tmp_t w = tmp_alloc(o, &o->blk);
  box_t bx; block_box(o, blk, &bx);
  unpack_even(o, in_abi, in);
  box_gather(o, &bx, in, bi, 0, NULL);
  A_block(o, &bx, bi, bo, w);
  box_gather(o, &bx, NULL, bo, 1, out);
  pack_even(o, out, out_abi);
  free(in); free(out); free(bi); free(bo); tmp_free(w);
}

void ora_apply_precond(ora_t *o, const double *r_abi, double *z_abi, int n_inner, int only_block) {
  size_t n = (size_t)o->Ls * o->V4 * 12;
  cplx *r = malloc(n * sizeof(cplx)), *z = malloc(n * sizeof(cplx));
  unpack_even(o, r_abi, r);
  precond_lat(o, r, z, n_inner, only_block);
  pack_even(o, z, z_abi);
  free(r); free(z);
}

typedef struct {
  int iters, reliable_updates, converged, breakdown;
  long inner_applies;
  double true_res, seconds;
} ora_stats;

/* ---- Algorithm 1 (r0 = b - A x0 first, R15), Polak-Ribiere beta eq. 18
 *       in the form of R16, fp64 throughout (no sloppy precision in Oracle-B). ---- */
int ora_solve(ora_t *o, const double *b_abi, double *x_abi, double tol, int max_iter, int use_precond,
              int n_inner, ora_stats *st, double *hist /* |r_k|/|b| for k = 1..nhist, may be NULL */, int nhist) {
  size_t n = (size_t)o->Ls * o->V4 * 12;
  cplx *b = malloc(n * sizeof(cplx)), *x = malloc(n * sizeof(cplx)), *r = malloc(n * sizeof(cplx));
  cplx *p = malloc(n * sizeof(cplx)), *z = malloc(n * sizeof(cplx)), *Ap = malloc(n * sizeof(cplx));
  tmp_t w = tmp_alloc(o, &o->lat);
  memset(st, 0, sizeof(*st));
  o->n_inner_applies = 0;
  double t0 = 0;
#ifdef _OPENMP
  t0 = omp_get_wtime();
#endif
  unpack_even(o, b_abi, b);
  unpack_even(o, x_abi, x); /* x0 */
  double bnorm = sqrt(rdot(n, b, b));
  if (bnorm == 0.0) {
    memset(x, 0, n * sizeof(cplx)); st->converged = 1;
  } else {
    MdagM_box(o, &o->lat, x, Ap, w);
    xmy(n, b, Ap, r);
    double rnorm = sqrt(rdot(n, r, r));
    if (rnorm <= tol * bnorm) st->converged = 1;
    else {
      if (use_precond) precond_lat(o, r, z, n_inner, -1); else memcpy(z, r, n * sizeof(cplx));
      memcpy(p, z, n * sizeof(cplx));
    }
    double rz = rdot(n, r, z);
    int k = 0;
    while (!st->converged && k < max_iter) {
      MdagM_box(o, &o->lat, p, Ap, w);
      double pAp = rdot(n, p, Ap);
      if (!(pAp > 0.0)) { st->breakdown = 1; break; }
      double alpha = rz / pAp;
      axpy(n, alpha, p, x);
      axpy(n, -alpha, Ap, r);
      rnorm = sqrt(rdot(n, r, r));
      k++;
      if (hist && k <= nhist) hist[k - 1] = rnorm / bnorm;
      int replaced = 0;
      if (rnorm <= tol * bnorm) { /* R15: confirm with the true residual */
        cplx *t = malloc(n * sizeof(cplx));
        MdagM_box(o, &o->lat, x, t, w);
        xmy(n, b, t, r);
        free(t);
        rnorm = sqrt(rdot(n, r, r));
        st->reliable_updates++;
        replaced = 1;
        if (rnorm <= tol * bnorm) { st->converged = 1; break; }
      }
      if (use_precond) precond_lat(o, r, z, n_inner, -1); else memcpy(z, r, n * sizeof(cplx));
      double rz2 = rdot(n, r, z);
      /* eq. 18: <z', r' - r>/<z, r> with r' - r = -alpha A p (the axpy above); Alg. 1's ratio right after a replacement (R16) */
      double beta = replaced ? rz2 / rz : -alpha * rdot(n, z, Ap) / rz;
#pragma omp parallel for schedule(static)
      for (long i = 0; i < (long)n; i++) p[i] = z[i] + beta * p[i];
      rz = rz2;
    }
    st->iters = k;
    MdagM_box(o, &o->lat, x, Ap, w);
    xmy(n, b, Ap, r);
    st->true_res = sqrt(rdot(n, r, r)) / bnorm;
  }
  pack_even(o, x, x_abi);
  st->inner_applies = o->n_inner_applies;
#ifdef _OPENMP
  st->seconds = omp_get_wtime() - t0;
#endif
  free(b); free(x); free(r); free(p); free(z); free(Ap); tmp_free(w);
  return st->converged ? 0 : (st->breakdown ? -6 : -5);
}

int ora_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
