// geometry.hpp -- host-side index tables of libmspcg (no CUDA).
//
// A "geometry" is what a hop stage needs to know about 4D sites, independent of Ls and of the gauge field:
//   * an E list (even sites) and an O list (odd sites) with their coordinates,
//   * for every list site its 8 neighbours as indices into the other list (or -1 = no contribution).
//
// Two geometries are built per context:
//   BLOCK  -- one Dirichlet block ("virtual node") with its snake-term halo: sites whose L1
//             overshoot d outside the block is <= 2 (even) / <= 1 (odd), the minimal site sets of PAPER.md:226
//             (Fig. 3; reading R11).  Local coordinates run over [-2, B+2) in cut directions (the padded box of
//             PAPER.md:224, reading R10 "PAD"); links are looked up by global periodic index.  Every block of the
//             lattice has the same tables; only the block origin differs.
//   FULL   -- the whole periodic lattice, sites ordered block-major (block b's interior even sites are the
//             contiguous range [b*nE0, (b+1)*nE0) in the same order as the BLOCK geometry's first nE0 sites), so a
//             block's part of a lattice vector is a contiguous sub-vector and the preconditioner needs no gather.
//
// Direction code: dir = 2*mu + 0 -> neighbour x+mu (term (1 - g_mu) U_mu(x) psi(x+mu) of PAPER.md:105 eq. 8),
//                 dir = 2*mu + 1 -> neighbour x-mu (term (1 + g_mu) U_mu(x-mu)^dag psi(x-mu)).
#pragma once
#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <vector>

namespace mspcg {

struct Geometry {
  int nblk = 0;        // blocks that share these tables (FULL: 1)
  int nE0 = 0;         // even sites with d = 0 (first nE0 entries of the E list)
  int nE = 0;          // E list length (BLOCK: even sites d <= 2; FULL: V4/2)
  int nO0 = 0;         // odd sites with d = 0
  int nO = 0;          // O list length (BLOCK: odd sites d <= 1; FULL: V4/2)
  std::vector<short> cE, cO;       // [n][4] coordinates: BLOCK = relative to the block origin, FULL = global
  std::vector<int> nbrE, nbrO;     // [n][8]: E-list site -> O-list index, O-list site -> E-list index
  std::vector<short> origin;       // [nblk][4] block origins (FULL: one zero origin)
};

struct Lattice {
  int L[4], B[4], nb[4], nblk;
  bool cut[4];
  long V4;
  Geometry blk, full;
  std::vector<int> e_int_to_cb;    // FULL E-list index -> ABI x_cb (even parity)
  std::vector<int> o_int_to_cb;    // FULL O-list index -> ABI x_cb (odd parity)
};

inline int pmod(int a, int m) { int r = a % m; return r < 0 ? r + m : r; }

inline void build_block_geometry(Lattice& lat) {
  Geometry& g = lat.blk;
  int ext[4], off[4];
  for (int d = 0; d < 4; d++) { ext[d] = lat.cut[d] ? lat.B[d] + 4 : lat.L[d]; off[d] = lat.cut[d] ? 2 : 0; }
  long nbox = (long)ext[0] * ext[1] * ext[2] * ext[3];
  std::vector<int> idx(nbox, -1);  // box lex -> list index (E or O by parity), -1 = not in a list
  auto overshoot = [&](const int c[4]) {
    int dsum = 0;
    for (int d = 0; d < 4; d++) if (lat.cut[d]) { if (c[d] < 0) dsum += -c[d]; else if (c[d] >= lat.B[d]) dsum += c[d] - lat.B[d] + 1; }
    return dsum;
  };
  // List order: interior (d = 0) sites first, then the halo; inside each part sites are ordered by 4x4x2x2 CELL (cells in
  // lexicographic order, x fastest) and lexicographically (x fastest) inside a cell, the same rule for both parities.  The
  // sites of one cell and parity are therefore one contiguous run of the list, and so are the rows and planes of a cell that a
  // neighbouring cell needs: the tile kernel (hop_tile.cuh, tile_tables.hpp) fetches a tile's inputs with few large copies.
  {
    const int cell[4] = {4, 4, 2, 2};
    struct Ent { int pass; long key; long lex; int par; };
    std::vector<Ent> ents;
    ents.reserve(nbox);
    for (long i = 0; i < nbox; i++) {
      long r = i; int c[4];
      for (int d = 0; d < 4; d++) { c[d] = (int)(r % ext[d]) - off[d]; r /= ext[d]; }
      const int par = pmod(c[0] + c[1] + c[2] + c[3], 2);
      const int dd = overshoot(c);
      if (!((par == 0 && dd <= 2) || (par == 1 && dd <= 1))) continue;
      long key = 0;
      for (int d = 3; d >= 0; d--) key = key * 4096 + (c[d] + 4) / cell[d];   // c >= -2, so c + 4 > 0 keeps cell 0 aligned at c = 0 (4 % cell == 0)
      ents.push_back({dd == 0 ? 0 : 1, key, i, par});
    }
    std::sort(ents.begin(), ents.end(), [](const Ent& a, const Ent& b) {
      if (a.pass != b.pass) return a.pass < b.pass;
      if (a.key != b.key) return a.key < b.key;
      return a.lex < b.lex;
    });
    for (const Ent& e : ents) {
      long r = e.lex; int c[4];
      for (int d = 0; d < 4; d++) { c[d] = (int)(r % ext[d]) - off[d]; r /= ext[d]; }
      if (e.par == 0) { idx[e.lex] = g.nE++; for (int d = 0; d < 4; d++) g.cE.push_back((short)c[d]); if (e.pass == 0) g.nE0 = g.nE; }
      else            { idx[e.lex] = g.nO++; for (int d = 0; d < 4; d++) g.cO.push_back((short)c[d]); if (e.pass == 0) g.nO0 = g.nO; }
    }
  }
  auto neighbours = [&](const std::vector<short>& cs, int n, std::vector<int>& out) {
    out.assign((size_t)n * 8, -1);
    for (int i = 0; i < n; i++)
      for (int mu = 0; mu < 4; mu++)
        for (int bw = 0; bw < 2; bw++) {
          int c[4] = {cs[4 * i], cs[4 * i + 1], cs[4 * i + 2], cs[4 * i + 3]};
          c[mu] += bw ? -1 : 1;
          if (lat.cut[mu]) { if (c[mu] < -2 || c[mu] >= lat.B[mu] + 2) continue; }  // zero Dirichlet at the pad edge
          else c[mu] = pmod(c[mu], lat.L[mu]);                                        // uncut: wraps inside the block
          long lex = 0;
          for (int d = 3; d >= 0; d--) lex = lex * ext[d] + (c[d] + off[d]);
          out[(size_t)i * 8 + 2 * mu + bw] = idx[lex];
        }
  };
  neighbours(g.cE, g.nE, g.nbrE);
  neighbours(g.cO, g.nO, g.nbrO);
  g.nblk = lat.nblk;
  g.origin.resize((size_t)lat.nblk * 4);
  for (int b = 0; b < lat.nblk; b++) {
    int r = b;
    for (int d = 0; d < 4; d++) { g.origin[4 * b + d] = (short)((r % lat.nb[d]) * lat.B[d]); r /= lat.nb[d]; }
  }
}

inline void build_full_geometry(Lattice& lat) {
  const Geometry& bg = lat.blk;
  Geometry& g = lat.full;
  long Vh = lat.V4 / 2;
  g.nblk = 1; g.nE0 = g.nE = (int)Vh; g.nO0 = g.nO = (int)Vh;
  g.origin.assign(4, 0);
  g.cE.resize((size_t)Vh * 4); g.cO.resize((size_t)Vh * 4);
  std::vector<int> lex2int(lat.V4, -1);
  lat.e_int_to_cb.resize(Vh); lat.o_int_to_cb.resize(Vh);
  auto lexof = [&](const int c[4]) { return c[0] + (long)lat.L[0] * (c[1] + (long)lat.L[1] * (c[2] + (long)lat.L[2] * c[3])); };
  for (int b = 0; b < lat.nblk; b++) {
    const short* o = &bg.origin[4 * b];
    for (int i = 0; i < bg.nE0; i++) {
      int c[4]; for (int d = 0; d < 4; d++) c[d] = o[d] + bg.cE[4 * i + d];
      long k = (long)b * bg.nE0 + i, lx = lexof(c);
      for (int d = 0; d < 4; d++) g.cE[4 * k + d] = (short)c[d];
      lex2int[lx] = (int)k; lat.e_int_to_cb[k] = (int)(lx / 2);
    }
    for (int i = 0; i < bg.nO0; i++) {
      int c[4]; for (int d = 0; d < 4; d++) c[d] = o[d] + bg.cO[4 * i + d];
      long k = (long)b * bg.nO0 + i;
      for (int d = 0; d < 4; d++) g.cO[4 * k + d] = (short)c[d];
      lex2int[lexof(c)] = (int)k; lat.o_int_to_cb[k] = (int)(lexof(c) / 2);
    }
  }
  auto neighbours = [&](const std::vector<short>& cs, long n, std::vector<int>& out) {
    out.resize((size_t)n * 8);
    for (long i = 0; i < n; i++)
      for (int mu = 0; mu < 4; mu++)
        for (int bw = 0; bw < 2; bw++) {
          int c[4] = {cs[4 * i], cs[4 * i + 1], cs[4 * i + 2], cs[4 * i + 3]};
          c[mu] = pmod(c[mu] + (bw ? -1 : 1), lat.L[mu]);
          out[(size_t)i * 8 + 2 * mu + bw] = lex2int[lexof(c)];
        }
  };
  neighbours(g.cE, Vh, g.nbrE);
  neighbours(g.cO, Vh, g.nbrO);
}

inline bool build_lattice(Lattice& lat, const int L[4], const int B[4]) {
  lat.V4 = 1; lat.nblk = 1;
  for (int d = 0; d < 4; d++) {
    if (L[d] < 2 || (L[d] & 1) || B[d] < 2 || (B[d] & 1) || L[d] % B[d] || L[d] > 4096) return false;
    lat.L[d] = L[d]; lat.B[d] = B[d]; lat.nb[d] = L[d] / B[d]; lat.cut[d] = B[d] != L[d];
    lat.V4 *= L[d]; lat.nblk *= lat.nb[d];
  }
  if (lat.V4 / 2 > 0x7fffffffL / 8) return false;
  build_block_geometry(lat);
  build_full_geometry(lat);
  return true;
}

// ---- Ls x Ls fifth-dimension matrices ("constant matrices diagonal in 4D"; readings R1, R3, R4) -----
// P+ block of  a*1 + d*S_minus,  (S_minus psi)_s = psi_{s-1}, (S_minus psi)_0 = -mf psi_{Ls-1};  P- block = transpose.
struct Mat { int n = 0; std::vector<double> a; double& at(int i, int j) { return a[(size_t)i * n + j]; } double at(int i, int j) const { return a[(size_t)i * n + j]; } };
inline Mat mat_bidiag(int Ls, double diag, double sub, double mf) {
  Mat m; m.n = Ls; m.a.assign((size_t)Ls * Ls, 0.0);
  for (int s = 0; s < Ls; s++) { m.at(s, s) += diag; if (s > 0) m.at(s, s - 1) += sub; else m.at(0, Ls - 1) += -mf * sub; }
  return m;
}
inline Mat mat_T(const Mat& x) { Mat m; m.n = x.n; m.a.resize(x.a.size()); for (int i = 0; i < x.n; i++) for (int j = 0; j < x.n; j++) m.at(i, j) = x.at(j, i); return m; }
inline Mat mat_mul(const Mat& x, const Mat& y) {
  Mat m; m.n = x.n; m.a.assign(x.a.size(), 0.0);
  for (int i = 0; i < x.n; i++) for (int k = 0; k < x.n; k++) { double v = x.at(i, k); if (v != 0.0) for (int j = 0; j < x.n; j++) m.at(i, j) += v * y.at(k, j); }
  return m;
}
// Inverse by Gauss-Jordan with partial pivoting (the matrix is strongly diagonally dominant: |alpha| >> |beta|).
inline bool mat_inv(const Mat& x, Mat& out) {
  int n = x.n; std::vector<long double> w((size_t)n * 2 * n, 0.0L);
  for (int i = 0; i < n; i++) { for (int j = 0; j < n; j++) w[(size_t)i * 2 * n + j] = x.at(i, j); w[(size_t)i * 2 * n + n + i] = 1.0L; }
  for (int col = 0; col < n; col++) {
    int piv = col; long double best = 0;
    for (int r = col; r < n; r++) { long double v = w[(size_t)r * 2 * n + col]; if (v < 0) v = -v; if (v > best) { best = v; piv = r; } }
    if (best == 0) return false;
    if (piv != col) for (int j = 0; j < 2 * n; j++) { long double t = w[(size_t)piv * 2 * n + j]; w[(size_t)piv * 2 * n + j] = w[(size_t)col * 2 * n + j]; w[(size_t)col * 2 * n + j] = t; }
    long double inv = 1.0L / w[(size_t)col * 2 * n + col];
    for (int j = 0; j < 2 * n; j++) w[(size_t)col * 2 * n + j] *= inv;
    for (int r = 0; r < n; r++) if (r != col) { long double f = w[(size_t)r * 2 * n + col]; if (f != 0) for (int j = 0; j < 2 * n; j++) w[(size_t)r * 2 * n + j] -= f * w[(size_t)col * 2 * n + j]; }
  }
  out.n = n; out.a.resize((size_t)n * n);
  for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) out.at(i, j) = (double)w[(size_t)i * 2 * n + n + j];
  return true;
}

}  // namespace mspcg
