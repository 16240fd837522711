// mspcg.cu -- C ABI of libmspcg (include/mspcg.h): context, workspace carving, kernel launch sequences for
// D^dag D (eq. 15-16), the multi-splitting preconditioner and the
// outer PCG with reliable updates (Algorithm 1, 283-289).  All arithmetic runs in the kernels of
// kernels.cuh; this file only sequences launches and moves scalars.  There is no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <type_traits>
#include <string>
#include <vector>

#include "../../include/mspcg.h"
#include "geometry.hpp"
#include <cuda_fp16.h>
#include "kernels.cuh"

using namespace mspcg;

namespace {

constexpr int KMAX = 32;  // most inner iterations per preconditioner application

struct Arena {
  char* base = nullptr; size_t off = 0; size_t cap = 0;
  template <typename T> T* take(size_t n) {
    off = (off + 255) & ~(size_t)255;
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
  void* take_bytes(size_t n) { return take<char>(n); }
};

struct GeomDev { int *nbrE = nullptr, *nbrO = nullptr; short *cE = nullptr, *cO = nullptr, *origin = nullptr; };
// Site tiles of the fp16 tile kernel (hop_tile.cuh) for the four stage launches of one geometry: kernel 2 (O list, inputs
// limited to the block interior), kernel 4 (O list), kernels 3 and 5 on the interior E sites, kernel 3 on the halo E sites.
struct TileSet {
  std::vector<TileRec> hO_lim, hO_all, hE_int, hE_halo;     // host
  TileRec *O_lim = nullptr, *O_all = nullptr, *E_int = nullptr, *E_halo = nullptr;   // device
  bool have = false;
};

// One set of fifth-dimension matrices (device, transposed per chirality: m[ch][s'][s]) in one compute type.
template <typename C> struct MatSet { C *K2 = nullptr, *K3a = nullptr, *K3b = nullptr, *K4 = nullptr, *K5 = nullptr, *K3h = nullptr; };
// The same matrices as fp16 mma.m16n8k16 A fragments [chirality 2][lane 32] (hop_mma.cuh).
struct MatFrag { uint4 *K2 = nullptr, *K3a = nullptr, *K3b = nullptr, *K4 = nullptr, *K5 = nullptr, *K3h = nullptr; };
struct HostMats { std::vector<double> K2, K3a, K3b, K4, K5, K3h; Mat A, F, Ainv; double diag, off; };

// Everything one precision needs to apply D^dag D on one geometry.
struct OpBuf {
  int prec = 0, ng = 18;
  void *linksE = nullptr, *linksO = nullptr; uint8_t *flipE = nullptr, *flipO = nullptr;
  void *t1 = nullptr, *tO = nullptr, *y = nullptr, *w = nullptr;  // [nblk*nE0], [nblk*nO], [nblk*nE0], [nblk*nE]
  bool have = false;
};

}  // namespace

struct mspcg_ctx {
  Lattice lat;
  int Ls = 0, Ls_hat = 0;
  double b = 0, c = 0, M5 = 0, mf = 0, alpha = 0, beta = 0, mu_shift = 0;
  HostMats hm, hm_hat;
  std::vector<double> T_host;
  std::string err;
  long launches = 0;
  int num_sms = 148;
  // optional per-launch CUDA-event timing (mspcg_timing): class = geometry*5 + kind
  bool timing = false; int cur_geom = 0;
  std::vector<cudaEvent_t> ev_pool; std::vector<int> ev_cls; size_t ev_used = 0;
  // configuration
  int outer_prec = 0, inner_prec = 0, recon = 18;
  bool configured = false, have_ws = false, have_gauge = false;
  size_t ws_bytes = 0;
  // device
  GeomDev gfull, gblk;
  TileSet tfull, tblk;
  bool dense_tma = true;         // mspcg_apply_M5inv through dense5d_tma.cuh (MSPCG_M5_TMA=0: the cp.async kernel of transfer_tc.cuh)
  int fixed_bits = 0;            // 8 / 16: fp32 inner CG vectors pass through the fixed-point store of eq. 17 (mspcg_set_fixed_storage); 0 = off
  int group_blocks = 0;          // Dirichlet blocks per L2-resident group of the preconditioner (0: all blocks at once); MSPCG_GROUP or mspcg_set_block_group
  bool use_tiles = true;         // MSPCG_TILE=0 in the environment selects the per-warp kernel k_hop_mma (A/B measurements)
  int *e_int_to_cb = nullptr, *o_int_to_cb = nullptr;   // FULL list index -> ABI x_cb, even / odd parity
  double* negI = nullptr;        // device [2][Ls][Ls]: minus the identity (full 2x2 operator of eq. 4, mspcg_apply_full)
  MatSet<double> md, md_hat; MatSet<float> mf32, mf32_hat; MatFrag mfr, mfr_hat;
  OpBuf full64, fullS, blkI;     // full lattice fp64 / sloppy; block geometry in the inner precision
  void *in_r = nullptr, *in_p = nullptr, *in_q = nullptr, *in_x = nullptr;   // inner CG vectors [V5h]
  double *rho = nullptr, *pq = nullptr; float* scale = nullptr; double* sc = nullptr;  // device scalars
  double* Tm = nullptr;          // device copy of the reduced-Ls transfer matrix T_host (A10)
  double* Gdev = nullptr;        // gradient accumulator of the T training (A12)
  float* BK2 = nullptr; uint4* fragI = nullptr;   // A/B of kernel 2 with the 5D matrix on tcgen05 (MSPCG_DENSE_TC=1): Mphi M5^-1 as [hi][s][s'], identity fragments
  bool dense_tc_ab = false;
  float* Bm5[2] = {nullptr, nullptr};        // chirality blocks of M5^-1 and M5^-dag (fp32 [hi][s][s']) for k_dense5d_tc
  __half *Bfwd = nullptr, *Bbwd = nullptr;   // fp16 B-operand images of T and T^dag for the tcgen05 transfer kernels
  bool transfer_tc = true;       // use them when (Ls, Ls_hat) is a compiled pair and the inner storage is fp16
  double* sc_host = nullptr;     // pinned
  double *v_b = nullptr, *v_xhi = nullptr, *v_rhi = nullptr, *v_t64 = nullptr;   // solver, fp64 native
  void *v_xlo = nullptr, *v_rlo = nullptr, *v_p = nullptr, *v_Ap = nullptr, *v_z = nullptr;  // solver, sloppy
  void *stage_in = nullptr, *stage_out = nullptr;   // native staging for ABI-layout calls (fp64-sized)
  double *abi_in = nullptr, *abi_out = nullptr;     // device ABI buffers for the *_host calls
};

cudaError_t dense5d_tma(mspcg_ctx* c, const void* in, void* out, const float* Mimg, long n_sites, int Ls, cudaStream_t st);

namespace {

int fail(mspcg_ctx* ctx, int code, const char* fmt, ...) {
  if (ctx) {
    char buf[512]; va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof(buf), fmt, ap); va_end(ap);
    ctx->err = buf;
  }
  return code;
}
#define CUDA_OK(ctx, expr)                                                                              \
  do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return fail(ctx, MSPCG_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)

bool ls_supported(int Ls) { return Ls == 4 || Ls == 6 || Ls == 8 || Ls == 12 || Ls == 16; }
bool prec_ok(int p) { return p == MSPCG_F64 || p == MSPCG_F32 || p == MSPCG_F16; }
long v5h(const mspcg_ctx* c, int Ls) { return c->lat.V4 / 2 * Ls; }
size_t vec_bytes(const mspcg_ctx* c, int prec, int Ls) { return (size_t)v5h(c, Ls) * 24 * prec; }

void transposed(const Mat& up, const Mat& lo, std::vector<double>& out) {
  int n = up.n; out.resize((size_t)2 * n * n);
  for (int s = 0; s < n; s++) for (int r = 0; r < n; r++) { out[(size_t)r * n + s] = up.at(s, r); out[(size_t)(n + r) * n + s] = lo.at(s, r); }
}
bool build_host_mats(HostMats& h, int Ls, double b, double c, double M5, double mf) {
  double alpha = b * (4.0 - M5) + 1.0, beta = c * (4.0 - M5) - 1.0;
  h.A = mat_bidiag(Ls, alpha, beta, mf);            // M5 on P+ (R3)
  h.F = mat_bidiag(Ls, -0.5 * b, -0.5 * c, mf);     // Mphi on P+ (R1, R3)
  if (!mat_inv(h.A, h.Ainv)) return false;
  h.diag = -0.5 * b; h.off = -0.5 * c;
  Mat At = mat_T(h.Ainv), Ft = mat_T(h.F);
  transposed(mat_mul(h.F, h.Ainv), mat_mul(Ft, At), h.K2);     // Mphi M5^-1           (kernel 2 of eq. 16)
  transposed(h.Ainv, At, h.K3a);                               // M5^-1                (kernel 3, first factor)
  transposed(At, h.Ainv, h.K3b);                               // M5^-dag              (kernel 3, second factor)
  transposed(mat_mul(At, Ft), mat_mul(h.Ainv, h.F), h.K4);     // M5^-dag Mphi^dag     (kernel 4)
  transposed(Ft, h.F, h.K5);                                   // Mphi^dag             (kernel 5)
  transposed(mat_mul(At, h.Ainv), mat_mul(h.Ainv, At), h.K3h); // - M5^-dag M5^-1      (kernel 3 on the halo sites of a Dirichlet block,
  for (double& v : h.K3h) v = -v;                              //                       where the xpay operand is zero: w = -M5^-dag M5^-1 D^w tO)
  return true;
}

// ------------------------------------------------------------------------------------------------ workspace carving
void carve_geom(Arena& a, GeomDev& g, const Geometry& h) {
  g.nbrE = a.take<int>(h.nbrE.size()); g.nbrO = a.take<int>(h.nbrO.size());
  g.cE = a.take<short>(h.cE.size()); g.cO = a.take<short>(h.cO.size()); g.origin = a.take<short>(h.origin.size());
}
template <typename C> void carve_mats(Arena& a, MatSet<C>& m, int Ls) {
  size_t n = (size_t)2 * Ls * Ls;
  m.K2 = a.take<C>(n); m.K3a = a.take<C>(n); m.K3b = a.take<C>(n); m.K4 = a.take<C>(n); m.K5 = a.take<C>(n); m.K3h = a.take<C>(n);
}
void carve_frags(Arena& a, MatFrag& m) {
  m.K2 = a.take<uint4>(64); m.K3a = a.take<uint4>(64); m.K3b = a.take<uint4>(64); m.K4 = a.take<uint4>(64); m.K5 = a.take<uint4>(64); m.K3h = a.take<uint4>(64);
}
void carve_links(Arena& a, OpBuf& o, const Geometry& g, int prec, int ng) {
  o.prec = prec; o.ng = ng; o.have = true;
  size_t nblk = g.nblk;
  o.linksE = a.take_bytes(nblk * g.nE * 8 * ng * prec); o.linksO = a.take_bytes(nblk * g.nO * 8 * ng * prec);
  o.flipE = a.take<uint8_t>(nblk * g.nE); o.flipO = a.take<uint8_t>(nblk * g.nO);
}
void carve_temps(Arena& a, OpBuf& o, const Geometry& g, int Ls) {   // stage vectors of eq. 16: live only inside one operator application
  size_t nblk = g.nblk, site = (size_t)Ls * 24 * o.prec;
  o.t1 = a.take_bytes(nblk * g.nE0 * site); o.tO = a.take_bytes(nblk * g.nO * site);
  o.y = a.take_bytes(nblk * g.nE0 * site); o.w = a.take_bytes(nblk * g.nE * site);
}
// Workspace layout.  Memory is sized for 180 GB at the largest configuration (48^3 x 96, Ls 12): buffers that are never live
// at the same time share storage --
//   * the stage vectors of the fp64 operator (used by residual replacements and fp64 applies) overlay the stage vectors of
//     the sloppy operator, of the block operator and the inner-CG vectors (none holds data between two calls);
//   * the staging buffers of the ABI-layout and *_host entry points overlay the solver's fp64 vectors (a solve and an apply
//     call never run at the same time on one context).
void carve_tiles(Arena& a, TileSet& t) {
  if (!t.have) return;
  t.O_lim = a.take<TileRec>(t.hO_lim.size()); t.O_all = a.take<TileRec>(t.hO_all.size());
  t.E_int = a.take<TileRec>(t.hE_int.size()); t.E_halo = a.take<TileRec>(t.hE_halo.size());
}
void build_tile_set(TileSet& t, const Geometry& g) {
  if (t.have) return;
  t.hO_lim = build_tiles(g.cO, g.nbrO, 0, g.nO, g.nE0);
  if (g.nE0 == g.nE) t.hO_all.clear(); else t.hO_all = build_tiles(g.cO, g.nbrO, 0, g.nO, g.nE);   // FULL: kernel 4 uses kernel 2's tiles
  t.hE_int = build_tiles(g.cE, g.nbrE, 0, g.nE0, g.nO);
  t.hE_halo = build_tiles(g.cE, g.nbrE, g.nE0, g.nE, g.nO);
  t.have = true;
}
void carve(mspcg_ctx* c, Arena& a) {
  const Lattice& L = c->lat;
  carve_geom(a, c->gfull, L.full); carve_geom(a, c->gblk, L.blk);
  carve_tiles(a, c->tfull); carve_tiles(a, c->tblk);
  c->e_int_to_cb = a.take<int>(L.e_int_to_cb.size()); c->o_int_to_cb = a.take<int>(L.o_int_to_cb.size());
  c->negI = a.take<double>((size_t)2 * c->Ls * c->Ls);
  carve_mats(a, c->md, c->Ls); carve_mats(a, c->mf32, c->Ls); carve_frags(a, c->mfr);
  for (int d = 0; d < 2; d++) c->Bm5[d] = a.take<float>((size_t)2 * c->Ls * c->Ls);
  c->BK2 = a.take<float>((size_t)2 * c->Ls * c->Ls); c->fragI = a.take<uint4>(64);
  if (c->Ls_hat) { carve_mats(a, c->md_hat, c->Ls_hat); carve_mats(a, c->mf32_hat, c->Ls_hat); carve_frags(a, c->mfr_hat); }
  c->rho = a.take<double>((size_t)(KMAX + 1) * L.nblk); c->pq = a.take<double>((size_t)KMAX * L.nblk);
  c->scale = a.take<float>(L.nblk); c->sc = a.take<double>(16);
  if (c->Ls_hat) { size_t nt = (size_t)4 * c->Ls_hat * 4 * c->Ls; c->Tm = a.take<double>(nt * 2); c->Bfwd = a.take<__half>(nt * 4); c->Bbwd = a.take<__half>(nt * 4); c->Gdev = a.take<double>(nt * 2); }
  carve_links(a, c->full64, L.full, MSPCG_F64, 18);
  if (c->outer_prec != MSPCG_F64) carve_links(a, c->fullS, L.full, c->outer_prec, c->recon);
  carve_links(a, c->blkI, L.blk, c->inner_prec, c->inner_prec == MSPCG_F64 ? 18 : c->recon);
  a.off = (a.off + 255) & ~(size_t)255;
  Arena u1 = a, u2 = a;                                   // two overlays of the same region
  carve_temps(u1, c->full64, L.full, c->Ls);
  if (c->outer_prec != MSPCG_F64) carve_temps(u2, c->fullS, L.full, c->Ls);
  carve_temps(u2, c->blkI, L.blk, c->Ls);
  size_t ni = vec_bytes(c, c->inner_prec, c->Ls);
  c->in_r = u2.take_bytes(ni); c->in_p = u2.take_bytes(ni); c->in_q = u2.take_bytes(ni);
  c->in_x = u2.take_bytes(vec_bytes(c, c->inner_prec == MSPCG_F64 ? MSPCG_F64 : MSPCG_F32, c->Ls));
  a.off = u1.off > u2.off ? u1.off : u2.off;
  size_t n64 = vec_bytes(c, MSPCG_F64, c->Ls), nS = vec_bytes(c, c->outer_prec, c->Ls);
  c->v_b = (double*)a.take_bytes(n64); c->v_xhi = (double*)a.take_bytes(n64); c->v_rhi = (double*)a.take_bytes(n64);
  c->v_t64 = (double*)a.take_bytes(n64);
  c->v_xlo = a.take_bytes(nS); c->v_rlo = a.take_bytes(nS); c->v_p = a.take_bytes(nS); c->v_Ap = a.take_bytes(nS);
  c->v_z = a.take_bytes(nS);
  c->stage_in = c->v_b; c->stage_out = c->v_xhi;
  c->abi_in = c->v_rhi; c->abi_out = c->v_t64;
}

// ------------------------------------------------------------------------------------------------ per-launch timing
enum { KIND_MPHI = 0, KIND_HOP_PLAIN = 1, KIND_HOP_K3 = 2, KIND_HOP_XPAY = 3, KIND_BLAS = 4, NKIND = 5, NCLASS = 10 };
struct TimedLaunch {   // records an event pair around one launch when timing is on
  mspcg_ctx* c; cudaStream_t st; bool on;
  TimedLaunch(mspcg_ctx* c_, int kind, cudaStream_t st_) : c(c_), st(st_), on(c_->timing) {
    if (!on) return;
    if (c->ev_used + 2 > c->ev_pool.size()) { cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b); c->ev_pool.push_back(a); c->ev_pool.push_back(b); }
    c->ev_cls.push_back(c->cur_geom * NKIND + kind);
    cudaEventRecord(c->ev_pool[c->ev_used], st);
  }
  ~TimedLaunch() { if (on) { cudaEventRecord(c->ev_pool[c->ev_used + 1], st); c->ev_used += 2; } }
};

// ------------------------------------------------------------------------------------------------ kernel launchers
#define DISPATCH_LS(LSV, ...)                                            \
  switch (LSV) {                                                         \
    case 4: { constexpr int LS = 4; __VA_ARGS__; } break;                \
    case 6: { constexpr int LS = 6; __VA_ARGS__; } break;                \
    case 8: { constexpr int LS = 8; __VA_ARGS__; } break;                \
    case 12: { constexpr int LS = 12; __VA_ARGS__; } break;              \
    default: { constexpr int LS = 16; __VA_ARGS__; } break;              \
  }

template <typename T, int LS, int EPI> size_t hop_smem() {
  typedef typename ST<T>::C C; typedef Smem<C, LS> SM;
  return sizeof(C) * ((size_t)SM::NS * SM::USTRIDE + (size_t)SM::NS * SM::SSTRIDE + (size_t)(EPI == EPI_K3 ? 4 : 2) * LS * LS) + sizeof(int) * SM::NS * 8;
}
template <typename T, int LS, int EPI>
cudaError_t launch_hop(mspcg_ctx* c, const HopArgs<T>& a, int nblk, cudaStream_t st, bool timed = true) {
  const bool was_timing = c->timing;
  if (!timed) c->timing = false;   // the caller times a group of launches as one (kernel 3 = interior + halo launch)
  const int kind = EPI == EPI_PLAIN ? KIND_HOP_PLAIN : (EPI == EPI_K3 ? KIND_HOP_K3 : KIND_HOP_XPAY);
  if constexpr (std::is_same<T, __half>::value) {   // fp16 storage: tensor-core kernels (hop_tile.cuh, hop_mma.cuh)
    if (a.tiles != nullptr && a.n_tiles > 0 && a.ng == 18) {   // thread-block-cooperative tile kernel
      static bool tattr = false;
      const size_t tsm = TileCfg<LS, EPI>::SMEM;
      if (!tattr) { cudaFuncSetAttribute(k_hop_tile<LS, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsm); tattr = true; }
      HopArgs<__half> ab = a; ab.nblk = nblk;
      const long total = (long)nblk * a.n_tiles;
      const unsigned grid = (unsigned)(total < c->num_sms ? total : c->num_sms);   // persistent: one thread block per SM
      { TimedLaunch tl(c, kind, st); k_hop_tile<LS, EPI><<<grid, TileCfg<LS, EPI>::THREADS, tsm, st>>>(ab); }
      c->launches++;
      c->timing = was_timing;
      return cudaPeekAtLastError();
    }
    constexpr int NW = MmaCfg<LS>::NW;
    static bool attr = false;
    const size_t sm = MmaSmem<LS>::BLOCK;
    if (!attr) {
      cudaFuncSetAttribute(k_hop_mma<LS, EPI, 18>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
      cudaFuncSetAttribute(k_hop_mma<LS, EPI, 12>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
      attr = true;
    }
    // persistent warps: one wave of <= 4 thread blocks per SM, over the sites of a Dirichlet block (grid.x) and over blocks (grid.y)
    const int slots = 4 * c->num_sms;
    int gx = (a.n_out + NW - 1) / NW, cap = slots / nblk;
    if (gx > cap) gx = cap;
    if (gx < 1) gx = 1;
    int gy = slots / gx; if (gy > nblk) gy = nblk; if (gy < 1) gy = 1;
    dim3 block(32 * NW), grid(gx, gy);
    HopArgs<__half> ab = a; ab.nblk = nblk;
    { TimedLaunch tl(c, kind, st);
      if (a.ng == 12) k_hop_mma<LS, EPI, 12><<<grid, block, sm, st>>>(ab); else k_hop_mma<LS, EPI, 18><<<grid, block, sm, st>>>(ab); }
  } else {
    static bool attr = false;
    const size_t sm = hop_smem<T, LS, EPI>();
    if (!attr) { cudaFuncSetAttribute(k_hop<T, LS, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); attr = true; }
    dim3 block(LS, Tile<LS>::NS), grid((a.n_out + Tile<LS>::NS - 1) / Tile<LS>::NS, nblk);
    { TimedLaunch tl(c, kind, st); k_hop<T, LS, EPI><<<grid, block, sm, st>>>(a); }
  }
  c->launches++;
  c->timing = was_timing;
  return cudaPeekAtLastError();
}
template <typename T, int LS>
cudaError_t launch_mphi(mspcg_ctx* c, const MphiArgs<T>& a, int nblk, cudaStream_t st) {
  typedef typename ST<T>::C C; typedef Smem<C, LS> SM;
  static bool attr = false;
  const size_t sm = sizeof(C) * (size_t)SM::NS * SM::SSTRIDE;
  if (!attr) { cudaFuncSetAttribute(k_mphi<T, LS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); attr = true; }
  dim3 block(LS, Tile<LS>::NS), grid((unsigned)((a.n_sites + Tile<LS>::NS - 1) / Tile<LS>::NS), nblk);
  { TimedLaunch tl(c, KIND_MPHI, st); k_mphi<T, LS><<<grid, block, sm, st>>>(a); }
  c->launches++;
  return cudaPeekAtLastError();
}

template <typename C> struct MatPick;
template <> struct MatPick<double> { static const MatSet<double>& get(const mspcg_ctx* c, bool hat) { return hat ? c->md_hat : c->md; } };
template <> struct MatPick<float> { static const MatSet<float>& get(const mspcg_ctx* c, bool hat) { return hat ? c->mf32_hat : c->mf32; } };

// Geometry view handed to the operator sequence: tables + per-precision buffers, possibly offset to one block.
template <typename T> struct OpView {
  int nblk, nE0, nE, nO, ng, Ls; bool hat;
  const int *nbrE, *nbrO;
  const T *linksE, *linksO; const uint8_t *flipE, *flipO;
  T *t1, *tO, *y, *w;
  const TileRec *tO_lim = nullptr, *tO_all = nullptr, *tE_int = nullptr, *tE_halo = nullptr;   // fp16 tile kernel
  int ntO_lim = 0, ntO_all = 0, ntE_int = 0, ntE_halo = 0;
};
template <typename T> OpView<T> make_view(const mspcg_ctx* c, const OpBuf& o, const Geometry& g, const GeomDev& gd, int Ls, bool hat) {
  OpView<T> v;
  const TileSet& ts = (&g == &c->lat.full) ? c->tfull : c->tblk;
  if (sizeof(T) == 2 && ts.have && c->use_tiles && o.ng == 18) {
    v.tO_lim = ts.O_lim; v.ntO_lim = (int)ts.hO_lim.size();
    v.tO_all = ts.hO_all.empty() ? ts.O_lim : ts.O_all; v.ntO_all = ts.hO_all.empty() ? (int)ts.hO_lim.size() : (int)ts.hO_all.size();
    v.tE_int = ts.E_int; v.ntE_int = (int)ts.hE_int.size();
    v.tE_halo = ts.E_halo; v.ntE_halo = (int)ts.hE_halo.size();
  }
  v.nblk = g.nblk; v.nE0 = g.nE0; v.nE = g.nE; v.nO = g.nO; v.ng = o.ng; v.Ls = Ls; v.hat = hat;
  v.nbrE = gd.nbrE; v.nbrO = gd.nbrO;
  v.linksE = (const T*)o.linksE; v.linksO = (const T*)o.linksO; v.flipE = o.flipE; v.flipO = o.flipO;
  v.t1 = (T*)o.t1; v.tO = (T*)o.tO; v.y = (T*)o.y; v.w = (T*)o.w;
  return v;
}
template <typename T> OpView<T> one_block(const OpView<T>& v, int blk) {
  OpView<T> o = v; o.nblk = 1;
  o.linksE = v.linksE + (size_t)blk * v.nE * 8 * v.ng; o.linksO = v.linksO + (size_t)blk * v.nO * 8 * v.ng;
  o.flipE = v.flipE + (size_t)blk * v.nE; o.flipO = v.flipO + (size_t)blk * v.nO;
  return o;
}

// q = D^dag D p on the view's geometry.  `mp` describes kernel 1 (Mphi, possibly fused with a p-update; its `t`,
// `n_sites`, matrix entries are filled here).  If dot_out != null: dot_out[blk] += Re<p, q>.
//   K1  t1 = Mphi p                              K2  tO = (Mphi M5^-1) D^w t1
//   K3  y = p - M5^-1 D^w tO ; w = M5^-dag y     K4  tO = (M5^-dag Mphi^dag) D^w^dag w
//   K5  q = y - Mphi^dag D^w^dag tO              (eq. 16; on a Dirichlet block the stage outputs live on
//                                                 the site sets d<=1, d<=2, d<=1, d=0 of PAPER.md:226)
template <typename T, int LS>
cudaError_t apply_normal(mspcg_ctx* c, const OpView<T>& v, MphiArgs<T> mp, const T* p, T* q, double* dot_out, cudaStream_t st) {
  typedef typename ST<T>::C C;
  const MatSet<C>& m = MatPick<C>::get(c, v.hat);
  const MatFrag& mf = v.hat ? c->mfr_hat : c->mfr;
  const HostMats& hm = v.hat ? c->hm_hat : c->hm;
  cudaError_t e;
  mp.t = v.t1; mp.n_sites = v.nE0; mp.diag = (C)hm.diag; mp.off = (C)hm.off; mp.mf = (C)c->mf;
  if ((e = launch_mphi<T, LS>(c, mp, v.nblk, st)) != cudaSuccess) return e;
  HopArgs<T> a;
  memset(&a, 0, sizeof(a));
  a.ng = v.ng;
  // K2
  a.in = v.t1; a.in_stride = v.nE0; a.n_in_limit = v.nE0; a.out = v.tO; a.out_stride = v.nO; a.n_out = v.nO;
  a.nbr = v.nbrO; a.links = v.linksO; a.flip = v.flipO; a.link_stride = v.nO; a.mat1 = m.K2; a.frag1 = mf.K2; a.sg = (C)1;
  a.tiles = v.tO_lim; a.n_tiles = v.ntO_lim;
  if (sizeof(T) == 2 && c->dense_tc_ab && !v.hat && a.tiles != nullptr && (LS == 8 || LS == 12 || LS == 16)) {
    // A/B (MSPCG_DENSE_TC=1): kernel 2 with its Ls x Ls matrix on tcgen05 instead of on register fragments inside the
    // hop -- the hop kernel runs with the identity matrix into the (larger) buffer w, then k_dense5d_tma applies Mphi M5^-1: one more
    // pass over the stage vector.  Timed as one kernel-2 launch.
    TimedLaunch tl(c, KIND_HOP_PLAIN, st);
    HopArgs<T> h = a; h.out = v.w; h.frag1 = c->fragI;
    if ((e = launch_hop<T, LS, EPI_PLAIN>(c, h, v.nblk, st, false)) != cudaSuccess) return e;
    if ((e = dense5d_tma(c, v.w, v.tO, c->BK2, (long)v.nblk * v.nO, LS, st)) != cudaSuccess) return e;
  } else
  if ((e = launch_hop<T, LS, EPI_PLAIN>(c, a, v.nblk, st)) != cudaSuccess) return e;
  // K3: on the interior sites (d = 0) y = p - M5^-1 D^w tO, w = M5^-dag y; on the halo sites of a Dirichlet block p = 0 and y is
  // not needed, so w = -(M5^-dag M5^-1) D^w tO is one contraction with the product matrix (a plain-epilogue launch on the site
  // range [nE0, nE)).  The two launches are timed as one kernel 3.
  a.in = v.tO; a.in_stride = v.nO; a.n_in_limit = v.nO; a.out = v.w; a.out_stride = v.nE; a.n_out = v.nE0;
  a.out2 = v.y; a.out2_stride = v.nE0; a.n_out2 = v.nE0; a.aux = p; a.aux_stride = v.nE0; a.n_aux = v.nE0;
  a.nbr = v.nbrE; a.links = v.linksE; a.flip = v.flipE; a.link_stride = v.nE; a.mat1 = m.K3a; a.mat2 = m.K3b; a.frag1 = mf.K3a; a.frag2 = mf.K3b;
  a.tiles = v.tE_int; a.n_tiles = v.ntE_int;
  {
    TimedLaunch tl(c, KIND_HOP_K3, st);
    if ((e = launch_hop<T, LS, EPI_K3>(c, a, v.nblk, st, false)) != cudaSuccess) return e;
    if (v.nE > v.nE0) {
      HopArgs<T> h = a;
      h.out = v.w + (size_t)v.nE0 * LS * 24; h.n_out = v.nE - v.nE0;
      h.out2 = nullptr; h.n_out2 = 0; h.aux = nullptr; h.n_aux = 0;
      h.nbr = v.nbrE + (size_t)v.nE0 * 8; h.links = v.linksE + (size_t)v.nE0 * 8 * v.ng; h.flip = v.flipE + v.nE0;
      h.mat1 = m.K3h; h.mat2 = nullptr; h.frag1 = mf.K3h; h.frag2 = nullptr;
      h.tiles = v.tE_halo; h.n_tiles = v.ntE_halo;
      if (h.tiles != nullptr && h.n_tiles > 0) { h.out = v.w; h.links = v.linksE; }   // the tile tables carry absolute list indices
      if ((e = launch_hop<T, LS, EPI_PLAIN>(c, h, v.nblk, st, false)) != cudaSuccess) return e;
    }
  }
  // K4
  a.in = v.w; a.in_stride = v.nE; a.n_in_limit = v.nE; a.out = v.tO; a.out_stride = v.nO; a.n_out = v.nO;
  a.out2 = nullptr; a.aux = nullptr; a.n_aux = 0; a.nbr = v.nbrO; a.links = v.linksO; a.flip = v.flipO; a.link_stride = v.nO;
  a.mat1 = m.K4; a.mat2 = nullptr; a.frag1 = mf.K4; a.frag2 = nullptr; a.sg = (C)-1;
  a.tiles = v.tO_all; a.n_tiles = v.ntO_all;
  if ((e = launch_hop<T, LS, EPI_PLAIN>(c, a, v.nblk, st)) != cudaSuccess) return e;
  // K5
  a.in = v.tO; a.in_stride = v.nO; a.n_in_limit = v.nO; a.out = q; a.out_stride = v.nE0; a.n_out = v.nE0;
  a.aux = v.y; a.aux_stride = v.nE0; a.n_aux = v.nE0; a.dotv = p; a.dotv_stride = v.nE0; a.dot_out = dot_out; a.dot_stride = 1;
  a.nbr = v.nbrE; a.links = v.linksE; a.flip = v.flipE; a.link_stride = v.nE; a.mat1 = m.K5; a.frag1 = mf.K5;
  a.tiles = v.tE_int; a.n_tiles = v.ntE_int;
  return launch_hop<T, LS, EPI_XPAY>(c, a, v.nblk, st);
}

template <typename T> MphiArgs<T> mphi_plain(const T* in) { MphiArgs<T> a; memset(&a, 0, sizeof(a)); a.in = in; a.mode = 0; return a; }

inline dim3 grid_sites(long n_sites, int Ls, int nblk, int threads = 128) { return dim3((unsigned)((n_sites * Ls + threads - 1) / threads), nblk); }

template <typename TA, typename TB>
cudaError_t convert(mspcg_ctx* c, const void* a, void* b, long n_sites, int Ls, int nblk, const float* scale, int invert, double factor, cudaStream_t st) {
  k_convert<TA, TB><<<grid_sites(n_sites, Ls, nblk), 128, 0, st>>>((const TA*)a, (TB*)b, n_sites, Ls, scale, invert, factor);
  c->launches++;
  return cudaPeekAtLastError();
}
cudaError_t convert_any(mspcg_ctx* c, const void* a, int pa, void* b, int pb, long n_sites, int Ls, cudaStream_t st, double factor = 1.0) {
#define CV(PA, TA, PB, TB) if (pa == PA && pb == PB) return convert<TA, TB>(c, a, b, n_sites, Ls, 1, nullptr, 0, factor, st);
  CV(8, double, 8, double) CV(8, double, 4, float) CV(8, double, 2, __half)
  CV(4, float, 8, double) CV(4, float, 4, float) CV(4, float, 2, __half)
  CV(2, __half, 8, double) CV(2, __half, 4, float) CV(2, __half, 2, __half)
#undef CV
  return cudaErrorInvalidValue;
}

// ---------------------------------------------------------------------------------------- the preconditioner (A7, A8)
// tcgen05 transfer kernels (transfer_tc.cuh) for the compiled (Ls, Ls_hat) pairs; false = not available, use the generic ones.
template <typename TIO>
bool launch_transfer_tc(mspcg_ctx* c, bool forward, const TransferArgs& ta, int Ls, int Lh, int nblk, cudaStream_t st) {
  dim3 grid((unsigned)((ta.n_sites + tc::TILE - 1) / tc::TILE), nblk);
#define TT(LSV, LHV)                                                                                                     \
  if (Ls == LSV && Lh == LHV) {                                                                                          \
    static bool attr = false;                                                                                            \
    if (!attr) {                                                                                                         \
      cudaFuncSetAttribute(k_reduce_begin_tc<TIO, LSV, LHV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TransferCfg<LSV, LHV>::SMEM); \
      cudaFuncSetAttribute(k_reduce_end_tc<TIO, LSV, LHV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TransferCfg<LHV, LSV>::SMEM);   \
      attr = true;                                                                                                       \
    }                                                                                                                    \
    if (forward) k_reduce_begin_tc<TIO, LSV, LHV><<<grid, 128, TransferCfg<LSV, LHV>::SMEM, st>>>(ta);                   \
    else k_reduce_end_tc<TIO, LSV, LHV><<<grid, 128, TransferCfg<LHV, LSV>::SMEM, st>>>(ta);                             \
    return true;                                                                                                         \
  }
  TT(8, 4) TT(12, 6) TT(12, 8) TT(16, 8) TT(16, 12)
#undef TT
  return false;
}
template <> bool launch_transfer_tc<__half>(mspcg_ctx*, bool, const TransferArgs&, int, int, int, cudaStream_t) { return false; }

// LS is the fifth-dimension extent of the inner iteration: Ls, or Ls_hat when `reduced` (then the right-hand side is
// T r, the operator is built from the Ls_hat matrices, and z = T^dag x + mu r; eq. 19-21).
template <typename TIO, typename T, int LS>
cudaError_t precond_impl(mspcg_ctx* c, const TIO* r_in_all, TIO* z_out_all, int k, bool reduced, cudaStream_t st) {
  typedef typename std::conditional<sizeof(T) == 8, double, float>::type TX;
  const Geometry& g = c->lat.blk;
  const int nblk = g.nblk;                 // also the stride of the per-block scalar arrays rho[it][nblk], pq[it][nblk]
  const OpView<T> vall = make_view<T>(c, c->blkI, g, c->gblk, LS, reduced);
  c->cur_geom = 1;
  cudaError_t e;
  if ((e = cudaMemsetAsync(c->rho, 0, sizeof(double) * (size_t)(KMAX + 1) * nblk, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(c->pq, 0, sizeof(double) * (size_t)KMAX * nblk, st)) != cudaSuccess) return e;
  if (sizeof(T) == 2) { if ((e = cudaMemsetAsync(c->scale, 0, sizeof(float) * nblk, st)) != cudaSuccess) return e; }
  // Block-resident inner CG ("L2-cache-bandwidth bound for GPUs with large cache"): the blocks are
  // independent (R13), so all k inner iterations are run for a GROUP of G blocks before the next group is touched.  The group's
  // vectors r, p, q, x and the stage vectors of eq. 16 live in the same G-block buffers for every group; with G chosen so that they
  // fit in the 126 MB L2, HBM sees r in, z out and the group's links once per iteration.  G = 0: all blocks in one group.
  const int G = (c->group_blocks > 0 && c->group_blocks < nblk) ? c->group_blocks : nblk;
  const size_t io_blk = (size_t)g.nE0 * c->Ls * 24;       // reals of one block's part of an I/O vector (full Ls)
  T *r = (T*)c->in_r, *p = (T*)c->in_p, *q = (T*)c->in_q; TX* x = (TX*)c->in_x;
  // with fp32 inner storage the CG vectors r, p, q = A p, x can be passed through the 8- / 16-bit fixed-point store of eq. 17
  // (mspcg_set_fixed_storage): the values are those of fixed-point storage, the bytes in HBM stay fp32 (a numerics mode, not a bandwidth one)
  const int fb = (sizeof(T) == 4 && !reduced) ? c->fixed_bits : 0;
  for (int g0 = 0; g0 < nblk; g0 += G) {
    const int gn = g0 + G <= nblk ? G : nblk - g0;
    const TIO* r_in = r_in_all + (size_t)g0 * io_blk;
    TIO* z_out = z_out_all + (size_t)g0 * io_blk;
    double *rho = c->rho + g0, *pq = c->pq + g0;
    OpView<T> v = vall; v.nblk = gn;
    v.linksE = vall.linksE + (size_t)g0 * vall.nE * 8 * vall.ng; v.linksO = vall.linksO + (size_t)g0 * vall.nO * 8 * vall.ng;
    v.flipE = vall.flipE + (size_t)g0 * vall.nE; v.flipO = vall.flipO + (size_t)g0 * vall.nO;
    const float* scale = nullptr;
    if (sizeof(T) == 2) {   // fp16 storage: rescale every block's right-hand side to max-abs 1 (R14)
      { TimedLaunch tl(c, KIND_BLAS, st); k_maxabs<TIO><<<grid_sites(g.nE0, c->Ls, gn), 128, 0, st>>>(r_in, g.nE0, c->Ls, c->scale + g0); }
      c->launches++;
      scale = c->scale + g0;
    }
    { TimedLaunch tl(c, KIND_BLAS, st);
      bool done = false;
      if (reduced && sizeof(T) == 2 && c->transfer_tc) {
        TransferArgs ta; memset(&ta, 0, sizeof(ta));
        ta.in = r_in; ta.out = r; ta.Bimg = c->Bfwd; ta.n_sites = g.nE0; ta.scale = scale; ta.rho0 = rho;
        done = launch_transfer_tc<TIO>(c, true, ta, c->Ls, LS, gn, st);
      }
      if (done) {}
      else if (reduced) k_reduce_begin<TIO, T><<<grid_sites(g.nE0, LS, gn), 128, 0, st>>>(r_in, r, g.nE0, c->Ls, LS, c->Tm, scale, rho);
      else k_pre_begin<TIO, T><<<grid_sites(g.nE0, LS, gn), 128, 0, st>>>(r_in, r, g.nE0, LS, scale, rho, fb); }
    c->launches++;
    for (int it = 0; it < k; it++) {
      MphiArgs<T> mp; memset(&mp, 0, sizeof(mp));
      mp.in = r; mp.p = p; mp.mode = 2; mp.it = it; mp.nblk = nblk; mp.rho = rho; mp.pq = pq; mp.fixed_bits = fb;
      if ((e = apply_normal<T, LS>(c, v, mp, p, q, pq + (size_t)it * nblk, st)) != cudaSuccess) return e;
      if (fb) {   // q = A p goes through the fixed-point store and <p, q> is taken from the stored values
        if ((e = cudaMemsetAsync(pq + (size_t)it * nblk, 0, sizeof(double) * gn, st)) != cudaSuccess) return e;
        TimedLaunch tl(c, KIND_BLAS, st);
        k_fixed_store_dot<T><<<grid_sites(g.nE0, LS, gn), 128, 0, st>>>(q, p, g.nE0, LS, fb, pq + (size_t)it * nblk);
        c->launches++;
      }
      { TimedLaunch tl(c, KIND_BLAS, st);
        k_inner_update<T, TX, TIO><<<grid_sites(g.nE0, LS, gn), 128, 0, st>>>(p, q, r, x, z_out, g.nE0, LS, it, nblk, (it == k - 1 && !reduced) ? 1 : 0,
                                                                              rho, pq, scale, fb); }
      c->launches++;
    }
    if (reduced) {
      { TimedLaunch tl(c, KIND_BLAS, st);
        bool done = false;
        if (sizeof(T) == 2 && c->transfer_tc) {
          TransferArgs ta; memset(&ta, 0, sizeof(ta));
          ta.in = x; ta.rin = r_in; ta.out = z_out; ta.Bimg = c->Bbwd; ta.n_sites = g.nE0; ta.scale = scale; ta.mu = c->mu_shift;
          done = launch_transfer_tc<TIO>(c, false, ta, c->Ls, LS, gn, st);
        }
        if (!done) k_reduce_end<TX, TIO><<<grid_sites(g.nE0, c->Ls, gn), 128, 0, st>>>(x, r_in, z_out, g.nE0, c->Ls, LS, c->Tm, scale, c->mu_shift); }
      c->launches++;
    }
  }
  return cudaPeekAtLastError();
}

template <typename TIO>
cudaError_t precond_dispatch(mspcg_ctx* c, const TIO* r, TIO* z, int k, bool reduced, cudaStream_t st) {
  const int Ls = reduced ? c->Ls_hat : c->Ls;
  switch (c->inner_prec) {
    case MSPCG_F64: DISPATCH_LS(Ls, return (precond_impl<TIO, double, LS>(c, r, z, k, reduced, st)));
    case MSPCG_F32: DISPATCH_LS(Ls, return (precond_impl<TIO, float, LS>(c, r, z, k, reduced, st)));
    default: DISPATCH_LS(Ls, return (precond_impl<TIO, __half, LS>(c, r, z, k, reduced, st)));
  }
  return cudaErrorInvalidValue;
}
cudaError_t precond_any(mspcg_ctx* c, const void* r, void* z, int io_prec, int k, bool reduced, cudaStream_t st) {
  if (io_prec == MSPCG_F64) return precond_dispatch<double>(c, (const double*)r, (double*)z, k, reduced, st);
  if (io_prec == MSPCG_F32) return precond_dispatch<float>(c, (const float*)r, (float*)z, k, reduced, st);
  return precond_dispatch<__half>(c, (const __half*)r, (__half*)z, k, reduced, st);
}

// ------------------------------------------------------------------------------------------- full-lattice D^dag D
template <typename T>
cudaError_t normal_full(mspcg_ctx* c, const OpBuf& ob, const T* p, T* q, MphiArgs<T> mp, double* dot_out, cudaStream_t st) {
  OpView<T> v = make_view<T>(c, ob, c->lat.full, c->gfull, c->Ls, false);
  c->cur_geom = 0;
  DISPATCH_LS(c->Ls, return (apply_normal<T, LS>(c, v, mp, p, q, dot_out, st)));
  return cudaErrorInvalidValue;
}
const OpBuf* full_buf(const mspcg_ctx* c, int prec) {
  if (prec == MSPCG_F64) return &c->full64;
  if (prec == c->outer_prec && c->fullS.have) return &c->fullS;
  return nullptr;
}
cudaError_t normal_full_any(mspcg_ctx* c, int prec, const void* p, void* q, double* dot_out, cudaStream_t st) {
  const OpBuf* ob = full_buf(c, prec);
  if (!ob) return cudaErrorInvalidValue;
  if (prec == MSPCG_F64) return normal_full<double>(c, *ob, (const double*)p, (double*)q, mphi_plain<double>((const double*)p), dot_out, st);
  if (prec == MSPCG_F32) return normal_full<float>(c, *ob, (const float*)p, (float*)q, mphi_plain<float>((const float*)p), dot_out, st);
  return normal_full<__half>(c, *ob, (const __half*)p, (__half*)q, mphi_plain<__half>((const __half*)p), dot_out, st);
}

template <typename TA>
cudaError_t pack_any_t(mspcg_ctx* c, const TA* abi, void* nat, int prec, int to_native, cudaStream_t st, int parity) {
  const long Vh = c->lat.V4 / 2;
  const int* table = parity ? c->o_int_to_cb : c->e_int_to_cb;
#define PK(TT) DISPATCH_LS(c->Ls, { dim3 block(LS, Tile<LS>::NS), grid((unsigned)((Vh + Tile<LS>::NS - 1) / Tile<LS>::NS)); \
    k_pack<TT, LS, TA><<<grid, block, 0, st>>>(abi, (TT*)nat, table, Vh, to_native); })
  if (prec == MSPCG_F64) PK(double) else if (prec == MSPCG_F32) PK(float) else PK(__half)
#undef PK
  c->launches++;
  return cudaPeekAtLastError();
}
cudaError_t pack_any(mspcg_ctx* c, const double* abi, void* nat, int prec, int to_native, cudaStream_t st, int parity = 0) {
  return pack_any_t<double>(c, abi, nat, prec, to_native, st, parity);
}

template <typename T>
cudaError_t build_links(mspcg_ctx* c, const double* U, OpBuf& o, const Geometry& g, const GeomDev& gd, int tb, cudaStream_t st) {
  const Lattice& L = c->lat;
  long nE = (long)g.nblk * g.nE, nO = (long)g.nblk * g.nO;
  k_build_links<T><<<(unsigned)((nE + 127) / 128), 128, 0, st>>>(U, (T*)o.linksE, o.flipE, gd.cE, gd.origin, g.nE, g.nblk, L.L[0], L.L[1], L.L[2], L.L[3], tb, o.ng);
  k_build_links<T><<<(unsigned)((nO + 127) / 128), 128, 0, st>>>(U, (T*)o.linksO, o.flipO, gd.cO, gd.origin, g.nO, g.nblk, L.L[0], L.L[1], L.L[2], L.L[3], tb, o.ng);
  c->launches += 2;
  return cudaPeekAtLastError();
}
cudaError_t build_links_any(mspcg_ctx* c, const double* U, OpBuf& o, const Geometry& g, const GeomDev& gd, int tb, cudaStream_t st) {
  if (o.prec == MSPCG_F64) return build_links<double>(c, U, o, g, gd, tb, st);
  if (o.prec == MSPCG_F32) return build_links<float>(c, U, o, g, gd, tb, st);
  return build_links<__half>(c, U, o, g, gd, tb, st);
}

template <typename C> cudaError_t upload_mats(const MatSet<C>& m, const HostMats& h, cudaStream_t st) {
  const std::vector<double>* src[6] = {&h.K2, &h.K3a, &h.K3b, &h.K4, &h.K5, &h.K3h};
  C* dst[6] = {m.K2, m.K3a, m.K3b, m.K4, m.K5, m.K3h};
  for (int i = 0; i < 6; i++) {
    std::vector<C> tmp(src[i]->begin(), src[i]->end());
    cudaError_t e = cudaMemcpyAsync(dst[i], tmp.data(), tmp.size() * sizeof(C), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    cudaStreamSynchronize(st);  // tmp goes out of scope
  }
  return cudaSuccess;
}
// fp16 A fragments of mma.m16n8k16 (row-major 16x16, zero padded) of the five matrices; src is the transposed-per-
// chirality array of build_host_mats: M_ch[s][s'] = src[(ch*n + s')*n + s].
cudaError_t upload_frags(const MatFrag& m, const HostMats& h, int n, cudaStream_t st) {
  const std::vector<double>* src[6] = {&h.K2, &h.K3a, &h.K3b, &h.K4, &h.K5, &h.K3h};
  uint4* dst[6] = {m.K2, m.K3a, m.K3b, m.K4, m.K5, m.K3h};
  for (int i = 0; i < 6; i++) {
    std::vector<uint32_t> tmp(2 * 32 * 4);
    auto M = [&](int ch, int s, int sp) -> float { return (s < n && sp < n) ? (float)(*src[i])[((size_t)ch * n + sp) * n + s] : 0.f; };
    auto h2 = [&](float lo, float hi) -> uint32_t {
      __half a = __float2half_rn(lo), b = __float2half_rn(hi); unsigned short ua, ub;
      memcpy(&ua, &a, 2); memcpy(&ub, &b, 2); return (uint32_t)ua | ((uint32_t)ub << 16);
    };
    for (int ch = 0; ch < 2; ch++)
      for (int lane = 0; lane < 32; lane++) {
        const int g = lane >> 2, t = lane & 3;
        uint32_t* q = &tmp[((size_t)ch * 32 + lane) * 4];
        q[0] = h2(M(ch, g, 2 * t), M(ch, g, 2 * t + 1));         q[1] = h2(M(ch, g + 8, 2 * t), M(ch, g + 8, 2 * t + 1));
        q[2] = h2(M(ch, g, 2 * t + 8), M(ch, g, 2 * t + 9));     q[3] = h2(M(ch, g + 8, 2 * t + 8), M(ch, g + 8, 2 * t + 9));
      }
    cudaError_t e = cudaMemcpyAsync(dst[i], tmp.data(), tmp.size() * 4, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    cudaStreamSynchronize(st);
  }
  return cudaSuccess;
}
template <typename V> cudaError_t up(void* dst, const std::vector<V>& src, cudaStream_t st) {
  return cudaMemcpyAsync(dst, src.data(), src.size() * sizeof(V), cudaMemcpyHostToDevice, st);
}

// The two chirality blocks of M5^-1 (d = 0) and M5^-dag (d = 1) for k_dense5d_tc, fp32 [hi][s][s']: on P+ (hi = 0) M5^-1 is A+^-1
// (hm.Ainv), on P- its transpose (R3); the dagger swaps them.  The kernel rounds to fp16 and builds the MMA's B operand itself.
int upload_m5_images(mspcg_ctx* ctx, cudaStream_t st) {
  const int Ls = ctx->Ls;
  for (int d = 0; d < 2; d++) {
    std::vector<float> m((size_t)2 * Ls * Ls);
    for (int hi = 0; hi < 2; hi++) for (int s = 0; s < Ls; s++) for (int sp = 0; sp < Ls; sp++)
      m[((size_t)hi * Ls + s) * Ls + sp] = (float)(((hi ^ d) == 0) ? ctx->hm.Ainv.at(s, sp) : ctx->hm.Ainv.at(sp, s));
    CUDA_OK(ctx, cudaMemcpyAsync(ctx->Bm5[d], m.data(), m.size() * sizeof(float), cudaMemcpyHostToDevice, st));
    CUDA_OK(ctx, cudaStreamSynchronize(st));
  }
  {  // kernel 2's matrix Mphi M5^-1 in the same form (hm.K2 is stored transposed per chirality: [ch][s'][s]) and identity fragments
    std::vector<float> m((size_t)2 * Ls * Ls);
    for (int hi = 0; hi < 2; hi++) for (int s = 0; s < Ls; s++) for (int sp = 0; sp < Ls; sp++)
      m[((size_t)hi * Ls + s) * Ls + sp] = (float)ctx->hm.K2[((size_t)hi * Ls + sp) * Ls + s];
    CUDA_OK(ctx, cudaMemcpyAsync(ctx->BK2, m.data(), m.size() * sizeof(float), cudaMemcpyHostToDevice, st));
    CUDA_OK(ctx, cudaStreamSynchronize(st));
    HostMats id; for (std::vector<double>* v : {&id.K2, &id.K3a, &id.K3b, &id.K4, &id.K5, &id.K3h}) { v->assign((size_t)2 * Ls * Ls, 0.0); for (int ch = 0; ch < 2; ch++) for (int i = 0; i < Ls; i++) (*v)[((size_t)ch * Ls + i) * Ls + i] = 1.0; }
    MatFrag mf; mf.K2 = mf.K3a = mf.K3b = mf.K4 = mf.K5 = mf.K3h = ctx->fragI;
    CUDA_OK(ctx, upload_frags(mf, id, Ls, st));
  }
  return MSPCG_OK;
}

// Device copies of the reduced-Ls transfer matrix: fp64 T for the generic kernels and the fp16 B-operand images of T and
// T^dag for the tcgen05 kernels (UMMA canonical K-major, no swizzle: element (n, k) at (n/8)*KG*64 + (k/8)*64 + (n%8)*8 + k%8).
int upload_T(mspcg_ctx* ctx, cudaStream_t st) {
  CUDA_OK(ctx, up(ctx->Tm, ctx->T_host, st)); CUDA_OK(ctx, cudaStreamSynchronize(st));
  const int Ls = ctx->Ls, Lh = ctx->Ls_hat;
  auto Tc = [&](int ah, int m, int s, int n, int ri) { return ctx->T_host[((((size_t)ah * 4 + m) * (4 * Ls)) + s * 4 + n) * 2 + ri]; };
  auto put = [&](std::vector<__half>& img, int KG, int n, int k, double v) { img[(size_t)(n / 8) * KG * 64 + (size_t)(k / 8) * 64 + (n % 8) * 8 + (k % 8)] = __float2half_rn((float)v); };
  std::vector<__half> f((size_t)64 * Ls * Lh), b((size_t)64 * Ls * Lh);
  for (int ah = 0; ah < Lh; ah++) for (int m = 0; m < 4; m++) for (int s = 0; s < Ls; s++) for (int n = 0; n < 4; n++) {
    const double tr = Tc(ah, m, s, n, 0), ti = Tc(ah, m, s, n, 1);
    // forward: row (ah, sp, hi, ri') with m = 2*hi + sp (fp16 fragment order), column (s, n, ri)
    const int rowf = ah * 8 + ((m & 1) * 2 + (m >> 1)) * 2, colf = s * 8 + n * 2;
    put(f, Ls, rowf, colf, tr); put(f, Ls, rowf, colf + 1, -ti); put(f, Ls, rowf + 1, colf, ti); put(f, Ls, rowf + 1, colf + 1, tr);
    // backward (conj T): row (s, n, ri'), column (ah, m, ri)
    const int rowb = s * 8 + n * 2, colb = ah * 8 + m * 2;
    put(b, Lh, rowb, colb, tr); put(b, Lh, rowb, colb + 1, ti); put(b, Lh, rowb + 1, colb, -ti); put(b, Lh, rowb + 1, colb + 1, tr);
  }
  CUDA_OK(ctx, up(ctx->Bfwd, f, st)); CUDA_OK(ctx, up(ctx->Bbwd, b, st)); CUDA_OK(ctx, cudaStreamSynchronize(st));
  return MSPCG_OK;
}

int check_ready(mspcg_ctx* c, bool need_gauge) {
  if (!c) return MSPCG_EINVAL;
  if (!c->have_ws) return fail(c, MSPCG_ENOWORKSPACE, "mspcg_set_workspace has not been called");
  if (need_gauge && !c->have_gauge) return fail(c, MSPCG_ENOGAUGE, "mspcg_load_gauge has not been called");
  return MSPCG_OK;
}

// scalar helpers for the outer loop: zero n device doubles / read them back synchronously
cudaError_t sc_zero(mspcg_ctx* c, int n, cudaStream_t st) { return cudaMemsetAsync(c->sc, 0, sizeof(double) * n, st); }
cudaError_t sc_read(mspcg_ctx* c, int n, cudaStream_t st) {
  cudaError_t e = cudaMemcpyAsync(c->sc_host, c->sc, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
  if (e != cudaSuccess) return e;
  return cudaStreamSynchronize(st);
}
template <typename T> cudaError_t dot2(mspcg_ctx* c, const T* a, const T* b, const T* cc, long nreal, cudaStream_t st, double* out = nullptr) {
  const long nchunk = nreal / ST<T>::PER;
  long blocks = (nchunk + 255) / 256; if (blocks > 148 * 16) blocks = 148 * 16;
  k_dot2<T><<<(unsigned)blocks, 256, 0, st>>>(a, b, cc, nchunk, out ? out : c->sc);
  c->launches++;
  return cudaPeekAtLastError();
}
template <typename T> cudaError_t axpby(mspcg_ctx* c, double a, const T* x, double b, T* y, long nreal, cudaStream_t st) {
  const long nchunk = nreal / ST<T>::PER;
  k_axpby<T><<<(unsigned)((nchunk + 255) / 256), 256, 0, st>>>(a, x, b, y, nchunk);
  c->launches++;
  return cudaPeekAtLastError();
}

// ------------------------------------------------------------------ full 4-step solve: set-up and tear-down
// fp64 on the FULL geometry.  PAPER.md:89-97: eq. (4) [[M5, M4eo],[M4oe, M5]](psi_e, psi_o) = (phi_e, phi_o), M4 = D^w Mphi (eq. 7).
template <int LS>
cudaError_t dense_full64(mspcg_ctx* c, const double* in, double* out, const double* mat, cudaStream_t st) {
  typedef Smem<double, LS> SM;
  static bool attr = false;
  const size_t sm = sizeof(double) * ((size_t)SM::NS * SM::SSTRIDE + (size_t)2 * LS * LS);
  if (!attr) { cudaFuncSetAttribute(k_dense5d<double, LS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); attr = true; }
  const long n = c->lat.V4 / 2;
  dim3 block(LS, Tile<LS>::NS), grid((unsigned)((n + Tile<LS>::NS - 1) / Tile<LS>::NS));
  k_dense5d<double, LS><<<grid, block, sm, st>>>(in, out, mat, n);
  c->launches++;
  return cudaPeekAtLastError();
}
// out = mat * D^w(^dag) in (EPI_PLAIN)  or  out = aux - mat * D^w(^dag) in (EPI_XPAY); to_odd: `in` on even sites, `out` on odd ones.
template <int LS, int EPI>
cudaError_t hop_full64(mspcg_ctx* c, const double* in, double* out, const double* aux, const double* mat, bool to_odd, double sg, cudaStream_t st) {
  const Geometry& g = c->lat.full; const OpBuf& o = c->full64;
  HopArgs<double> a; memset(&a, 0, sizeof(a));
  a.ng = o.ng; a.in = in; a.in_stride = g.nE; a.n_in_limit = g.nE; a.out = out; a.out_stride = g.nE; a.n_out = g.nE;
  a.aux = aux; a.aux_stride = g.nE; a.n_aux = aux ? g.nE : 0;
  a.nbr = to_odd ? c->gfull.nbrO : c->gfull.nbrE; a.links = (const double*)(to_odd ? o.linksO : o.linksE); a.flip = to_odd ? o.flipO : o.flipE;
  a.link_stride = g.nE; a.mat1 = mat; a.sg = sg;
  return launch_hop<double, LS, EPI>(c, a, 1, st);
}
template <int LS>
cudaError_t bidiag_full64(mspcg_ctx* c, const double* in, double* out, double diag, double off, cudaStream_t st) {
  MphiArgs<double> mp = mphi_plain<double>(in);
  mp.t = out; mp.n_sites = c->lat.V4 / 2; mp.diag = diag; mp.off = off; mp.mf = c->mf;
  return launch_mphi<double, LS>(c, mp, 1, st);
}
// phihat_e = M5^-1 phi_e - M5^-1 M4eo M5^-1 phi_o (eq. 6) -> hat;  rhs = D^dag phihat_e (eq. 9).  pe, po, hat, rhs: NATIVE fp64.
template <int LS>
cudaError_t prepare_source_impl(mspcg_ctx* c, const double* pe, const double* po, double* hat, double* rhs, cudaStream_t st) {
  const MatSet<double>& m = c->md; const OpBuf& o = c->full64;
  double *t1 = (double*)o.t1, *tO = (double*)o.tO, *w = (double*)o.w;
  cudaError_t e;
  if ((e = dense_full64<LS>(c, po, tO, m.K2, st)) != cudaSuccess) return e;                                  // Mphi M5^-1 phi_o
  if ((e = dense_full64<LS>(c, pe, t1, m.K3a, st)) != cudaSuccess) return e;                                 // M5^-1 phi_e
  if ((e = hop_full64<LS, EPI_XPAY>(c, tO, hat, t1, m.K3a, false, 1.0, st)) != cudaSuccess) return e;        // - M5^-1 D^w (.)
  if ((e = dense_full64<LS>(c, hat, w, m.K3b, st)) != cudaSuccess) return e;                                 // D^dag: M5^-dag
  if ((e = hop_full64<LS, EPI_PLAIN>(c, w, tO, nullptr, m.K4, true, -1.0, st)) != cudaSuccess) return e;     //   (M5^-dag Mphi^dag) D^w^dag
  return hop_full64<LS, EPI_XPAY>(c, tO, rhs, hat, m.K5, false, -1.0, st);                                   //   1 - Mphi^dag D^w^dag (.)
}
// psi_o = M5^-1 (phi_o - M4oe psi_e) (second row of eq. 4).  NATIVE fp64.
template <int LS>
cudaError_t reconstruct_odd_impl(mspcg_ctx* c, const double* xe, const double* po, double* xo, cudaStream_t st) {
  const MatSet<double>& m = c->md; const OpBuf& o = c->full64;
  double *t1 = (double*)o.t1, *w = (double*)o.w;
  cudaError_t e;
  if ((e = bidiag_full64<LS>(c, xe, t1, c->hm.diag, c->hm.off, st)) != cudaSuccess) return e;                // Mphi psi_e
  if ((e = dense_full64<LS>(c, po, w, m.K3a, st)) != cudaSuccess) return e;                                  // M5^-1 phi_o
  return hop_full64<LS, EPI_XPAY>(c, t1, xo, w, m.K3a, true, 1.0, st);                                       // - M5^-1 D^w (.)
}
// (out_e, out_o) = the 2x2 operator of eq. 4 on (psi_e, psi_o).  NATIVE fp64.
template <int LS>
cudaError_t apply_full_impl(mspcg_ctx* c, const double* xe, const double* xo, double* oe, double* oo, cudaStream_t st) {
  const OpBuf& o = c->full64;
  double *t1 = (double*)o.t1, *y = (double*)o.y;
  cudaError_t e;
  for (int par = 0; par < 2; par++) {   // out_par = M5 psi_par + D^w Mphi psi_other
    const double *same = par ? xo : xe, *other = par ? xe : xo;
    if ((e = bidiag_full64<LS>(c, same, y, c->alpha, c->beta, st)) != cudaSuccess) return e;
    if ((e = bidiag_full64<LS>(c, other, t1, c->hm.diag, c->hm.off, st)) != cudaSuccess) return e;
    if ((e = hop_full64<LS, EPI_XPAY>(c, t1, par ? oo : oe, y, c->negI, par != 0, 1.0, st)) != cudaSuccess) return e;
  }
  return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------ outer PCG (A11)
#define SOLVE_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return fail(c, MSPCG_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)

template <typename TS>
int solve_impl(mspcg_ctx* c, const double* b_abi, double* x_abi, const mspcg_solve_params* prm, mspcg_solve_stats* stt, cudaStream_t st) {
  const int Ls = c->Ls;
  const long nreal = v5h(c, Ls) * 24;
  const long Vh = c->lat.V4 / 2;
  const bool sloppy = sizeof(TS) != 8;
  const int sp = (int)sizeof(TS);
  const OpBuf& obS = sloppy ? c->fullS : c->full64;
  double *b = c->v_b, *xhi = c->v_xhi, *rhi = c->v_rhi, *t64 = c->v_t64;
  TS *xlo = (TS*)c->v_xlo, *rlo = (TS*)c->v_rlo, *p = (TS*)c->v_p, *Ap = (TS*)c->v_Ap;
  TS* z = prm->use_precond ? (TS*)c->v_z : rlo;
  memset(stt, 0, sizeof(*stt));
  const long launches0 = c->launches;
  cudaEvent_t ev0, ev1;
  SOLVE_CUDA(cudaEventCreate(&ev0)); SOLVE_CUDA(cudaEventCreate(&ev1));
  SOLVE_CUDA(cudaEventRecord(ev0, st));
  SOLVE_CUDA(pack_any(c, b_abi, b, MSPCG_F64, 1, st));
  SOLVE_CUDA(pack_any(c, x_abi, xhi, MSPCG_F64, 1, st));
  SOLVE_CUDA(sc_zero(c, 16, st));
  SOLVE_CUDA(dot2<double>(c, b, b, nullptr, nreal, st, c->sc + 8));
  SOLVE_CUDA(sc_read(c, 16, st));
  const double bnorm = std::sqrt(c->sc_host[8]);
  int k = 0, rc = MSPCG_OK;
  auto true_residual = [&](double* rn) -> cudaError_t {   // rhi = b - A xhi in fp64; *rn = |rhi|
    cudaError_t e;
    if ((e = normal_full<double>(c, c->full64, xhi, t64, mphi_plain<double>(xhi), nullptr, st)) != cudaSuccess) return e;
    stt->outer_applies++;
    if ((e = cudaMemcpyAsync(rhi, b, sizeof(double) * nreal, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return e;
    if ((e = axpby<double>(c, -1.0, t64, 1.0, rhi, nreal, st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(c->sc + 8, 0, sizeof(double), st)) != cudaSuccess) return e;
    if ((e = dot2<double>(c, rhi, rhi, nullptr, nreal, st, c->sc + 8)) != cudaSuccess) return e;
    if ((e = sc_read(c, 16, st)) != cudaSuccess) return e;
    *rn = std::sqrt(c->sc_host[8]);
    return cudaSuccess;
  };
  if (bnorm == 0.0) {  // R15: b = 0 -> x = 0
    SOLVE_CUDA(cudaMemsetAsync(x_abi, 0, sizeof(double) * nreal, st));
    stt->converged = 1;
  } else {
    double rnorm = 0, maxr;
    SOLVE_CUDA(true_residual(&rnorm));                       // r0 = b - A x0 (R15)
    // fp16 sloppy vectors are kept in units of sigma ~ |r| at the last residual replacement (r_lo = r_hi / sigma, so
    // x_lo = x_true / sigma, p likewise): alpha and beta are scale invariant, and fp16 never underflows as r shrinks.
    const bool rescale = sizeof(TS) == 2;
    const double unit = 16.0 / std::sqrt((double)nreal);   // |r_lo| = sqrt(n)/16: rms element 2^-4, three decades above the fp16 normal minimum
    double sigma = (rescale && rnorm > 0) ? rnorm * unit : 1.0;
    SOLVE_CUDA(convert_any(c, rhi, 8, rlo, sp, Vh, Ls, st, 1.0 / sigma));
    SOLVE_CUDA(cudaMemsetAsync(xlo, 0, sizeof(TS) * nreal, st));
    maxr = rnorm;
    if (rnorm <= prm->tol * bnorm) stt->converged = 1;
    else {
      if (prm->use_precond) { SOLVE_CUDA(precond_any(c, rlo, z, sp, prm->n_inner, prm->use_reduced_ls != 0, st)); stt->inner_applies += (long)prm->n_inner * c->lat.nblk; }
      SOLVE_CUDA(cudaMemcpyAsync(p, z, sizeof(TS) * nreal, cudaMemcpyDeviceToDevice, st));   // p0 = z0
      SOLVE_CUDA(sc_zero(c, SC_N, st));
      SOLVE_CUDA(dot2<TS>(c, rlo, z, nullptr, nreal, st, c->sc + SC_RZN));
    }
    // The loop keeps <z,r>, alpha and beta in device memory (k_outer_update, k_outer_scalars): no kernel waits for the host.  The host
    // reads (<p,Ap>, |r|^2) of iteration k - 1 from a pinned ring, written by the last kernel of that iteration, after it has queued
    // iteration k: convergence and the reliable-update rule (R17) are evaluated one iteration late, and the GPU never idles.
    constexpr int RING = 8;
    double* ring = c->sc_host + 16;
    cudaEvent_t evs[RING];
    for (int i = 0; i < RING; i++) SOLVE_CUDA(cudaEventCreateWithFlags(&evs[i], cudaEventDisableTiming));
    const bool self_z = !prm->use_precond;
    int ignore_upto = 0;             // snapshots of iterations <= this were taken before the last residual replacement
    auto replace_residual = [&]() -> int {   // R17 residual replacement / R15 confirmation with the true residual, then z, <z,r>, beta anew
      SOLVE_CUDA(convert_any(c, xlo, sp, t64, 8, Vh, Ls, st));
      SOLVE_CUDA(axpby<double>(c, sigma, t64, 1.0, xhi, nreal, st));
      SOLVE_CUDA(cudaMemsetAsync(xlo, 0, sizeof(TS) * nreal, st));
      SOLVE_CUDA(true_residual(&rnorm));
      double f2 = 1.0;
      if (rescale && rnorm > 0) {   // new unit: p keeps its true size, <z,r> follows
        const double f = sigma / (rnorm * unit);
        SOLVE_CUDA(axpby<TS>(c, 0.0, p, f, p, nreal, st));
        f2 = f * f; sigma = rnorm * unit;
      }
      SOLVE_CUDA(convert_any(c, rhi, 8, rlo, sp, Vh, Ls, st, 1.0 / sigma));
      maxr = rnorm; stt->reliable_updates++;
      if (rnorm <= prm->tol * bnorm) { stt->converged = 1; return MSPCG_OK; }
      if (prm->use_precond) { SOLVE_CUDA(precond_any(c, rlo, z, sp, prm->n_inner, prm->use_reduced_ls != 0, st)); stt->inner_applies += (long)prm->n_inner * c->lat.nblk; }
      SOLVE_CUDA(dot2<TS>(c, z, rlo, nullptr, nreal, st, c->sc + SC_RZN));
      k_outer_scalars<<<1, 1, 0, st>>>(c->sc, nullptr, 2, f2); c->launches++;
      return MSPCG_OK;
    };
    auto handle = [&](int it) -> int {   // look at the snapshot of iteration `it` (1-based)
      SOLVE_CUDA(cudaEventSynchronize(evs[it % RING]));
      const double pAp = ring[2 * (it % RING)], rr = ring[2 * (it % RING) + 1];
      const double rn = std::sqrt(rr) * sigma;
      if (it > ignore_upto) {
        if (!(pAp > 0.0) || !(rn == rn)) { stt->breakdown = 1; rc = MSPCG_EBREAKDOWN; return MSPCG_OK; }   // the update kernel used alpha = 0
        rnorm = rn;
      }
      if (prm->history && it <= prm->history_len) prm->history[it - 1] = rn / bnorm;
      if (it <= ignore_upto) return MSPCG_OK;
      if (rnorm <= prm->tol * bnorm || (sloppy && rnorm < prm->delta * maxr)) {
        ignore_upto = k;
        return replace_residual();
      }
      if (rnorm > maxr) maxr = rnorm;
      return MSPCG_OK;
    };
    int handled = 0;
    if (!stt->converged) { k_outer_scalars<<<1, 1, 0, st>>>(c->sc, nullptr, 3, 1.0); c->launches++; }
    while (!stt->converged && rc == MSPCG_OK && k < prm->max_iter) {
      // Ap = A p; for k > 0 the update p = z + beta p is fused into kernel 1 (beta read from device memory)
      MphiArgs<TS> mp; memset(&mp, 0, sizeof(mp));
      if (k == 0) { mp.in = p; mp.mode = 0; } else { mp.in = z; mp.p = p; mp.mode = 1; mp.beta_dev = c->sc + SC_BETA; }
      SOLVE_CUDA(normal_full<TS>(c, obS, p, Ap, mp, c->sc + SC_PAP, st));
      stt->outer_applies++;
      { const long nchunk = nreal / ST<TS>::PER;              // alpha_k = <r_k,z_k>/<p_k,A p_k> is formed on the device
        k_outer_update<TS><<<(unsigned)((nchunk + 255) / 256), 256, 0, st>>>(p, Ap, rlo, xlo, nchunk, c->sc, self_z ? 1 : 0);
        c->launches++; }
      k++;
      if (prm->use_precond) {
        SOLVE_CUDA(precond_any(c, rlo, z, sp, prm->n_inner, prm->use_reduced_ls != 0, st)); stt->inner_applies += (long)prm->n_inner * c->lat.nblk;
        SOLVE_CUDA(dot2<TS>(c, z, rlo, Ap, nreal, st, c->sc + SC_RZN));
      }
      k_outer_scalars<<<1, 1, 0, st>>>(c->sc, ring + 2 * (k % RING), 0, 1.0); c->launches++;   // eq. 18; snapshot for the host
      SOLVE_CUDA(cudaEventRecord(evs[k % RING], st));
      while (handled < k - 1 && !stt->converged && rc == MSPCG_OK) { handled++; int r_ = handle(handled); if (r_) return r_; }
    }
    while (handled < k && !stt->converged && rc == MSPCG_OK) { handled++; int r_ = handle(handled); if (r_) return r_; }
    for (int i = 0; i < RING; i++) cudaEventDestroy(evs[i]);
    if (!stt->converged && rc == MSPCG_OK) rc = MSPCG_ENOCONV;
    // x = x_hi + sigma x_lo, true residual, unpack
    SOLVE_CUDA(convert_any(c, xlo, sp, t64, 8, Vh, Ls, st));
    SOLVE_CUDA(axpby<double>(c, sigma, t64, 1.0, xhi, nreal, st));
    double rn = 0;
    SOLVE_CUDA(true_residual(&rn));
    stt->outer_applies--;   // the closing residual check is bookkeeping, not part of the iteration
    stt->true_res = rn / bnorm;
    SOLVE_CUDA(pack_any(c, x_abi, xhi, MSPCG_F64, 0, st));
  }
  stt->iters = k;
  SOLVE_CUDA(cudaEventRecord(ev1, st));
  SOLVE_CUDA(cudaEventSynchronize(ev1));
  float ms = 0; cudaEventElapsedTime(&ms, ev0, ev1);
  stt->seconds = ms * 1e-3;
  cudaEventDestroy(ev0); cudaEventDestroy(ev1);
  (void)launches0;
  return rc == MSPCG_OK ? MSPCG_OK : fail(c, rc, rc == MSPCG_ENOCONV ? "max_iter reached" : "breakdown: <p,Ap> <= 0 or NaN");
}

}  // namespace

// ------------------------------------------------------------------------------------------- training of T (A12)
// w = (+)_s A_s v on fp64 NATIVE vectors, through the block operator in the inner precision T (double: in place).
template <typename T>
cudaError_t block_operator64(mspcg_ctx* c, const double* v, double* w, cudaStream_t st) {
  const Geometry& g = c->lat.blk;
  OpView<T> view = make_view<T>(c, c->blkI, g, c->gblk, c->Ls, false);
  c->cur_geom = 1;
  const long Vh = c->lat.V4 / 2;
  cudaError_t e;
  if (sizeof(T) == 8) {
    DISPATCH_LS(c->Ls, return (apply_normal<T, LS>(c, view, mphi_plain<T>((const T*)v), (const T*)v, (T*)w, nullptr, st)));
  }
  if ((e = convert_any(c, v, 8, c->in_p, (int)sizeof(T), Vh, c->Ls, st)) != cudaSuccess) return e;
  DISPATCH_LS(c->Ls, e = (apply_normal<T, LS>(c, view, mphi_plain<T>((const T*)c->in_p), (const T*)c->in_p, (T*)c->in_q, nullptr, st)));
  if (e != cudaSuccess) return e;
  return convert_any(c, c->in_q, (int)sizeof(T), w, 8, Vh, c->Ls, st);
}

// chi2 = sum_i |M (T^dag Ahat T + mu) v_i - v_i|^2 and (optionally) G = d chi2 / d conj(T) = sum_i (c_i v_i^dag + a_i g_i^dag),
// e = M w - v, g = M e, a = Ahat T v, c = Ahat T g (eq. 22; reading R20).
template <typename T>
int train_eval_impl(mspcg_ctx* c, const double* v_abi, int nvec, int k, double* chi2, double* grad_host, cudaStream_t st) {
  typedef typename std::conditional<sizeof(T) == 8, double, float>::type TX;
  const int Ls = c->Ls, Lh = c->Ls_hat;
  const long Vh = c->lat.V4 / 2, nreal = v5h(c, Ls) * 24;
  const size_t nG = (size_t)16 * Lh * Ls * 2;
  struct NoGroups { mspcg_ctx* c; int g; NoGroups(mspcg_ctx* c_) : c(c_), g(c_->group_blocks) { c->group_blocks = 0; } ~NoGroups() { c->group_blocks = g; } } no_groups(c);   // in_x must hold every block
  double *V = (double*)c->stage_in, *W = (double*)c->stage_out, *E = c->v_t64, *Gv = c->v_rhi;
  const int spb = 32;
  const unsigned oblocks = (unsigned)((Vh + spb - 1) / spb);
  const size_t osm = sizeof(double) * 24 * (Ls + Lh);
  SOLVE_CUDA(cudaMemsetAsync(c->Gdev, 0, sizeof(double) * nG, st));
  SOLVE_CUDA(sc_zero(c, 2, st));
  for (int i = 0; i < nvec; i++) {
    SOLVE_CUDA(pack_any(c, v_abi + (size_t)i * nreal, V, MSPCG_F64, 1, st));
    SOLVE_CUDA(precond_dispatch<double>(c, V, W, k, true, st));                       // W = (T^dag Ahat T + mu) V ; in_x = a
    SOLVE_CUDA(block_operator64<T>(c, W, E, st));
    SOLVE_CUDA(axpby<double>(c, -1.0, V, 1.0, E, nreal, st));                          // e = M w - v
    SOLVE_CUDA(dot2<double>(c, E, E, nullptr, nreal, st));                             // chi2 += |e|^2 (accumulates in sc[0])
    if (grad_host) {
      SOLVE_CUDA(block_operator64<T>(c, E, Gv, st));                                   // g = M e
      k_outer_T<TX><<<oblocks, 512, osm, st>>>((const TX*)c->in_x, Gv, Vh, Ls, Lh, spb, c->Gdev); c->launches++;
      SOLVE_CUDA(precond_dispatch<double>(c, Gv, W, k, true, st));                     // in_x = c = Ahat T g
      k_outer_T<TX><<<oblocks, 512, osm, st>>>((const TX*)c->in_x, V, Vh, Ls, Lh, spb, c->Gdev); c->launches++;
      SOLVE_CUDA(cudaPeekAtLastError());
    }
  }
  SOLVE_CUDA(sc_read(c, 1, st));
  *chi2 = c->sc_host[0];
  if (grad_host) { SOLVE_CUDA(cudaMemcpyAsync(grad_host, c->Gdev, sizeof(double) * nG, cudaMemcpyDeviceToHost, st)); SOLVE_CUDA(cudaStreamSynchronize(st)); }
  return MSPCG_OK;
}

// Minimiser over the sampled interval of the quartic through five equally spaced points (exact line search when Ahat is
// linear; not trusted outside the interval because the fixed-count CG is only approximately linear):
// fit by elimination, cubic derivative solved in closed form.
double quartic_argmin(const double eta[5], const double val[5]) {
  double A[5][6];
  const double sc = eta[4] != 0 ? eta[4] : 1.0;   // work in x = eta / eta_max
  for (int i = 0; i < 5; i++) { double x = eta[i] / sc, p = 1; for (int j = 0; j < 5; j++) { A[i][j] = p; p *= x; } A[i][5] = val[i]; }
  for (int col = 0; col < 5; col++) {
    int piv = col; for (int r = col + 1; r < 5; r++) if (std::fabs(A[r][col]) > std::fabs(A[piv][col])) piv = r;
    for (int j = 0; j < 6; j++) std::swap(A[col][j], A[piv][j]);
    for (int r = 0; r < 5; r++) if (r != col) { double f = A[r][col] / A[col][col]; for (int j = col; j < 6; j++) A[r][j] -= f * A[col][j]; }
  }
  double cf[5]; for (int i = 0; i < 5; i++) cf[i] = A[i][5] / A[i][i];           // val = sum cf[j] x^j
  auto P = [&](double x) { return (((cf[4] * x + cf[3]) * x + cf[2]) * x + cf[1]) * x + cf[0]; };
  // derivative 4 c4 x^3 + 3 c3 x^2 + 2 c2 x + c1 = 0
  double a3 = 4 * cf[4], a2 = 3 * cf[3], a1 = 2 * cf[2], a0 = cf[1];
  double roots[3]; int nr = 0;
  if (std::fabs(a3) < 1e-300) {
    if (std::fabs(a2) > 1e-300) { double disc = a1 * a1 - 4 * a2 * a0; if (disc >= 0) { roots[nr++] = (-a1 + std::sqrt(disc)) / (2 * a2); roots[nr++] = (-a1 - std::sqrt(disc)) / (2 * a2); } }
    else if (std::fabs(a1) > 1e-300) roots[nr++] = -a0 / a1;
  } else {
    double b = a2 / a3, cc = a1 / a3, d = a0 / a3;
    double p = cc - b * b / 3, q = 2 * b * b * b / 27 - b * cc / 3 + d, disc = q * q / 4 + p * p * p / 27;
    if (disc > 0) { double sq = std::sqrt(disc); roots[nr++] = std::cbrt(-q / 2 + sq) + std::cbrt(-q / 2 - sq) - b / 3; }
    else { double r = std::sqrt(-p * p * p / 27), phi = std::acos(std::fmax(-1.0, std::fmin(1.0, -q / (2 * (r > 0 ? r : 1e-300))))), m = 2 * std::sqrt(-p / 3);
      for (int j = 0; j < 3; j++) roots[nr++] = m * std::cos((phi + 2 * M_PI * j) / 3) - b / 3; }
  }
  // minimiser of the fit over the sampled interval: stationary points inside [0, 1] and the sample points themselves
  double bx = 0.0, bv = P(0.0);
  for (int i = 1; i < 5; i++) { const double x = eta[i] / sc; if (P(x) < bv) { bv = P(x); bx = x; } }
  for (int j = 0; j < nr; j++) if (roots[j] >= 0.0 && roots[j] <= 1.0 && P(roots[j]) < bv) { bv = P(roots[j]); bx = roots[j]; }
  return bx * sc;
}

// out = (Ls x Ls chirality blocks Mimg) in on fp16 NATIVE vectors of n_sites site columns: tensor-map TMA + tcgen05 (dense5d_tma.cuh).
// cudaErrorNotSupported: Ls not compiled or the driver entry point is missing.
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                    const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static PFN_encodeTiled encode_tiled_fn() {
  static PFN_encodeTiled fn = nullptr; static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr; cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = (PFN_encodeTiled)p;
  }
  return fn;
}
// 4D map of an fp16 NATIVE vector with the dimension order (16-byte chunk, site, s, colour): see dense5d_tma.cuh
static bool native_f16_map(CUtensorMap* m, const void* base, long n_sites, int Ls) {
  PFN_encodeTiled enc = encode_tiled_fn();
  if (!enc) return false;
  const cuuint64_t dims[4] = {8, (cuuint64_t)n_sites, (cuuint64_t)Ls, 3};
  const cuuint64_t strides[3] = {(cuuint64_t)Ls * 48, 48, 16};
  const cuuint32_t box[4] = {8, 128, (cuuint32_t)Ls, 3}, estr[4] = {1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
cudaError_t dense5d_tma(mspcg_ctx* c, const void* in, void* out, const float* Mimg, long n_sites, int Ls, cudaStream_t st) {
  CUtensorMap mi, mo;
  if (!native_f16_map(&mi, in, n_sites, Ls) || !native_f16_map(&mo, out, n_sites, Ls)) return cudaErrorNotSupported;
  Dense5dTmaArgs a; a.M = Mimg; a.n_sites = n_sites;
  const long n_tiles = (n_sites + 127) / 128;
  const unsigned grid = (unsigned)(n_tiles < c->num_sms ? n_tiles : c->num_sms);
#define DT(LSV)                                                                                                            \
  if (Ls == LSV) {                                                                                                         \
    static bool attr = false;                                                                                              \
    if (!attr) { cudaFuncSetAttribute(k_dense5d_tma<LSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Dense5dTmaCfg<LSV>::SMEM); attr = true; } \
    k_dense5d_tma<LSV><<<grid, Dense5dTmaCfg<LSV>::THREADS, Dense5dTmaCfg<LSV>::SMEM, st>>>(mi, mo, a);                  \
    c->launches++;                                                                                                         \
    return cudaPeekAtLastError();                                                                                          \
  }
  DT(8) DT(12) DT(16)
#undef DT
  return cudaErrorNotSupported;
}

// ================================================================================================== C ABI
extern "C" {

int mspcg_create(mspcg_ctx** out, int Lx, int Ly, int Lz, int Lt, int Ls, double b, double c, double M5, double mf,
                 int Bx, int By, int Bz, int Bt) {
  if (!out) return MSPCG_EINVAL;
  *out = nullptr;
  if (!ls_supported(Ls)) return MSPCG_EINVAL;
  if (b * (4.0 - M5) + 1.0 == 0.0) return MSPCG_EINVAL;
  mspcg_ctx* ctx = new (std::nothrow) mspcg_ctx();
  if (!ctx) return MSPCG_ENOMEM;
  const int L[4] = {Lx, Ly, Lz, Lt}, B[4] = {Bx, By, Bz, Bt};
  if (!build_lattice(ctx->lat, L, B)) { delete ctx; return MSPCG_EINVAL; }
  ctx->Ls = Ls; ctx->b = b; ctx->c = c; ctx->M5 = M5; ctx->mf = mf;
  { const char* e = getenv("MSPCG_TRANSFER_TC"); if (e && e[0] == '0') ctx->transfer_tc = false; }
  { const char* e = getenv("MSPCG_TILE"); if (e && e[0] == '0') ctx->use_tiles = false; }
  { const char* e = getenv("MSPCG_GROUP"); if (e) ctx->group_blocks = atoi(e); }
  { const char* e = getenv("MSPCG_M5_TMA"); if (e && e[0] == '0') ctx->dense_tma = false; }
  { const char* e = getenv("MSPCG_DENSE_TC"); if (e && e[0] == '1') ctx->dense_tc_ab = true; }             // A/B switch: per-warp hop kernel   // debugging switch: generic transfer kernels
  ctx->alpha = b * (4.0 - M5) + 1.0; ctx->beta = c * (4.0 - M5) - 1.0;
  if (!build_host_mats(ctx->hm, Ls, b, c, M5, mf)) { delete ctx; return MSPCG_EINVAL; }
  *out = ctx;
  return MSPCG_OK;
}

int mspcg_destroy(mspcg_ctx* ctx) {
  if (!ctx) return MSPCG_EINVAL;
  if (ctx->sc_host) cudaFreeHost(ctx->sc_host);
  for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
  delete ctx;
  return MSPCG_OK;
}

const char* mspcg_last_error(const mspcg_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int mspcg_geometry(const mspcg_ctx* ctx, long out[5]) {
  if (!ctx || !out) return MSPCG_EINVAL;
  out[0] = ctx->lat.nblk; out[1] = ctx->lat.blk.nE0; out[2] = ctx->lat.blk.nE; out[3] = ctx->lat.blk.nO; out[4] = ctx->lat.V4 / 2;
  return MSPCG_OK;
}

int mspcg_get_matrix(const mspcg_ctx* ctx, int which, double* out_host) {
  if (!ctx || !out_host || which < 0 || which > 2) return MSPCG_EINVAL;
  const Mat& m = which == 0 ? ctx->hm.A : which == 1 ? ctx->hm.F : ctx->hm.Ainv;
  memcpy(out_host, m.a.data(), m.a.size() * sizeof(double));
  return MSPCG_OK;
}

int mspcg_set_reduced_ls(mspcg_ctx* ctx, int Ls_hat, const double* T_host, double mu) {
  if (!ctx) return MSPCG_EINVAL;
  if (ctx->configured) return fail(ctx, MSPCG_EINVAL, "mspcg_set_reduced_ls must precede mspcg_workspace_bytes");
  if (!ls_supported(Ls_hat) || Ls_hat > ctx->Ls || !T_host) return fail(ctx, MSPCG_EINVAL, "unsupported Ls_hat");
  if (!build_host_mats(ctx->hm_hat, Ls_hat, ctx->b, ctx->c, ctx->M5, ctx->mf)) return fail(ctx, MSPCG_EINVAL, "singular M5 at Ls_hat");
  ctx->Ls_hat = Ls_hat; ctx->mu_shift = mu;
  ctx->T_host.assign(T_host, T_host + (size_t)4 * Ls_hat * 4 * ctx->Ls * 2);
  return MSPCG_OK;
}

int mspcg_workspace_bytes(mspcg_ctx* ctx, int outer_prec, int inner_prec, int recon, size_t* bytes) {
  if (!ctx || !bytes) return MSPCG_EINVAL;
  if (!prec_ok(outer_prec) || !prec_ok(inner_prec) || (recon != 18 && recon != 12)) return fail(ctx, MSPCG_EINVAL, "bad precision or recon");
  if (ctx->have_ws) return fail(ctx, MSPCG_EINVAL, "workspace already set");
  ctx->outer_prec = outer_prec; ctx->inner_prec = inner_prec; ctx->recon = recon; ctx->configured = true;
  if (ctx->use_tiles && recon == 18) {   // site tiles of the fp16 tile kernel, for the geometries that run in fp16
    if (inner_prec == MSPCG_F16) build_tile_set(ctx->tblk, ctx->lat.blk);
    if (outer_prec == MSPCG_F16) build_tile_set(ctx->tfull, ctx->lat.full);
  }
  Arena a;
  carve(ctx, a);
  ctx->ws_bytes = (a.off + 255) & ~(size_t)255;
  *bytes = ctx->ws_bytes;
  return MSPCG_OK;
}

int mspcg_set_workspace(mspcg_ctx* ctx, void* workspace_dev, size_t bytes, void* stream) {
  if (!ctx) return MSPCG_EINVAL;
  if (!ctx->configured) return fail(ctx, MSPCG_EINVAL, "call mspcg_workspace_bytes first");
  if (!workspace_dev || bytes < ctx->ws_bytes || ((uintptr_t)workspace_dev & 255)) return fail(ctx, MSPCG_EINVAL, "workspace too small or misaligned");
  cudaStream_t st = (cudaStream_t)stream;
  Arena a; a.base = (char*)workspace_dev; a.cap = bytes;
  carve(ctx, a);
  const Lattice& L = ctx->lat;
  CUDA_OK(ctx, up(ctx->gfull.nbrE, L.full.nbrE, st)); CUDA_OK(ctx, up(ctx->gfull.nbrO, L.full.nbrO, st));
  CUDA_OK(ctx, up(ctx->gfull.cE, L.full.cE, st)); CUDA_OK(ctx, up(ctx->gfull.cO, L.full.cO, st));
  CUDA_OK(ctx, up(ctx->gfull.origin, L.full.origin, st));
  CUDA_OK(ctx, up(ctx->gblk.nbrE, L.blk.nbrE, st)); CUDA_OK(ctx, up(ctx->gblk.nbrO, L.blk.nbrO, st));
  CUDA_OK(ctx, up(ctx->gblk.cE, L.blk.cE, st)); CUDA_OK(ctx, up(ctx->gblk.cO, L.blk.cO, st));
  CUDA_OK(ctx, up(ctx->gblk.origin, L.blk.origin, st));
  CUDA_OK(ctx, up(ctx->e_int_to_cb, L.e_int_to_cb, st)); CUDA_OK(ctx, up(ctx->o_int_to_cb, L.o_int_to_cb, st));
  for (TileSet* t : {&ctx->tfull, &ctx->tblk}) {
    if (!t->have) continue;
    if (!t->hO_lim.empty()) CUDA_OK(ctx, up(t->O_lim, t->hO_lim, st));
    if (!t->hO_all.empty()) CUDA_OK(ctx, up(t->O_all, t->hO_all, st));
    if (!t->hE_int.empty()) CUDA_OK(ctx, up(t->E_int, t->hE_int, st));
    if (!t->hE_halo.empty()) CUDA_OK(ctx, up(t->E_halo, t->hE_halo, st));
  }
  { std::vector<double> ni((size_t)2 * ctx->Ls * ctx->Ls, 0.0);
    for (int ch = 0; ch < 2; ch++) for (int i = 0; i < ctx->Ls; i++) ni[((size_t)ch * ctx->Ls + i) * ctx->Ls + i] = -1.0;
    CUDA_OK(ctx, up(ctx->negI, ni, st)); }
  CUDA_OK(ctx, cudaStreamSynchronize(st));
  CUDA_OK(ctx, upload_mats<double>(ctx->md, ctx->hm, st)); CUDA_OK(ctx, upload_mats<float>(ctx->mf32, ctx->hm, st));
  CUDA_OK(ctx, upload_frags(ctx->mfr, ctx->hm, ctx->Ls, st));
  { int rc_ = upload_m5_images(ctx, st); if (rc_) return rc_; }
  if (ctx->Ls_hat) {
    CUDA_OK(ctx, upload_mats<double>(ctx->md_hat, ctx->hm_hat, st)); CUDA_OK(ctx, upload_mats<float>(ctx->mf32_hat, ctx->hm_hat, st));
    CUDA_OK(ctx, upload_frags(ctx->mfr_hat, ctx->hm_hat, ctx->Ls_hat, st));
    { int rc_ = upload_T(ctx, st); if (rc_) return rc_; }
  }
  if (!ctx->sc_host) CUDA_OK(ctx, cudaMallocHost(&ctx->sc_host, sizeof(double) * 64));
  { int dev = 0, n = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0) ctx->num_sms = n; }
  ctx->have_ws = true;
  return MSPCG_OK;
}

int mspcg_load_gauge(mspcg_ctx* ctx, const double* U_dev, int t_boundary, void* stream) {
  int rc = check_ready(ctx, false); if (rc) return rc;
  if (!U_dev || (t_boundary != 1 && t_boundary != -1)) return fail(ctx, MSPCG_EINVAL, "bad gauge pointer or t_boundary");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_OK(ctx, build_links_any(ctx, U_dev, ctx->full64, ctx->lat.full, ctx->gfull, t_boundary, st));
  if (ctx->fullS.have) CUDA_OK(ctx, build_links_any(ctx, U_dev, ctx->fullS, ctx->lat.full, ctx->gfull, t_boundary, st));
  CUDA_OK(ctx, build_links_any(ctx, U_dev, ctx->blkI, ctx->lat.blk, ctx->gblk, t_boundary, st));
  ctx->have_gauge = true;
  return MSPCG_OK;
}

size_t mspcg_vec_bytes(const mspcg_ctx* ctx, int prec) { return (ctx && prec_ok(prec)) ? vec_bytes(ctx, prec, ctx->Ls) : 0; }

int mspcg_pack(mspcg_ctx* ctx, const double* abi_dev, void* native_dev, int prec, void* stream) {
  int rc = check_ready(ctx, false); if (rc) return rc;
  if (!abi_dev || !native_dev || !prec_ok(prec)) return fail(ctx, MSPCG_EINVAL, "bad argument");
  CUDA_OK(ctx, pack_any(ctx, abi_dev, native_dev, prec, 1, (cudaStream_t)stream));
  return MSPCG_OK;
}
int mspcg_unpack(mspcg_ctx* ctx, const void* native_dev, double* abi_dev, int prec, void* stream) {
  int rc = check_ready(ctx, false); if (rc) return rc;
  if (!abi_dev || !native_dev || !prec_ok(prec)) return fail(ctx, MSPCG_EINVAL, "bad argument");
  CUDA_OK(ctx, pack_any(ctx, abi_dev, const_cast<void*>(native_dev), prec, 0, (cudaStream_t)stream));
  return MSPCG_OK;
}

int mspcg_apply_M5inv(mspcg_ctx* ctx, const void* in_dev, void* out_dev, int dagger, void* stream) {
  int rc = check_ready(ctx, false); if (rc) return rc;
  if (!in_dev || !out_dev || in_dev == out_dev) return fail(ctx, MSPCG_EINVAL, "bad pointer or aliasing");
  cudaStream_t st = (cudaStream_t)stream;
  if (ctx->dense_tma) {   // tensor-map TMA + tcgen05 kernel (dense5d_tma.cuh); MSPCG_M5_TMA=0 selects the cp.async kernel below
    cudaError_t e = dense5d_tma(ctx, in_dev, out_dev, ctx->Bm5[dagger ? 1 : 0], (long)(v5h(ctx, ctx->Ls) / ctx->Ls), ctx->Ls, st);
    if (e == cudaSuccess) return MSPCG_OK;
    if (e != cudaErrorNotSupported) return fail(ctx, MSPCG_ECUDA, "k_dense5d_tma: %s", cudaGetErrorString(e));
  }
  Dense5dTcArgs a;
  a.in = reinterpret_cast<const uint4*>(in_dev); a.out = reinterpret_cast<uint4*>(out_dev);
  a.M = ctx->Bm5[dagger ? 1 : 0]; a.n_sites = (long)(v5h(ctx, ctx->Ls) / ctx->Ls);
  const long n_tiles = (a.n_sites + tc::TILE - 1) / tc::TILE;
  const unsigned grid = (unsigned)(n_tiles < 2L * ctx->num_sms ? n_tiles : 2L * ctx->num_sms);   // persistent: two thread blocks per SM
#define DT(LSV)                                                                                                          \
  if (ctx->Ls == LSV) {                                                                                                  \
    static bool attr = false;                                                                                            \
    if (!attr) { cudaFuncSetAttribute(k_dense5d_tc<LSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Dense5dTcCfg<LSV>::SMEM); attr = true; } \
    k_dense5d_tc<LSV><<<grid, 128, Dense5dTcCfg<LSV>::SMEM, st>>>(a);                                                \
    ctx->launches++;                                                                                                     \
    CUDA_OK(ctx, cudaPeekAtLastError());                                                                                 \
    return MSPCG_OK;                                                                                                     \
  }
  DT(8) DT(12) DT(16)
#undef DT
  return fail(ctx, MSPCG_EINVAL, "mspcg_apply_M5inv: Ls must be 8, 12 or 16");
}

int mspcg_apply_MdagM(mspcg_ctx* ctx, const void* in_dev, void* out_dev, int prec, int layout, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!in_dev || !out_dev || in_dev == out_dev || !full_buf(ctx, prec)) return fail(ctx, MSPCG_EINVAL, "bad pointer, aliasing, or precision not configured");
  cudaStream_t st = (cudaStream_t)stream;
  if (layout == MSPCG_LAYOUT_NATIVE) {
    CUDA_OK(ctx, normal_full_any(ctx, prec, in_dev, out_dev, nullptr, st));
  } else {
    CUDA_OK(ctx, pack_any(ctx, (const double*)in_dev, ctx->stage_in, prec, 1, st));
    CUDA_OK(ctx, normal_full_any(ctx, prec, ctx->stage_in, ctx->stage_out, nullptr, st));
    CUDA_OK(ctx, pack_any(ctx, (double*)out_dev, ctx->stage_out, prec, 0, st));
  }
  return MSPCG_OK;
}

int mspcg_apply_precond(mspcg_ctx* ctx, const void* r_dev, void* z_dev, int io_prec, int layout, int n_inner,
                        int use_reduced, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!r_dev || !z_dev || n_inner < 1 || n_inner > KMAX || !prec_ok(io_prec)) return fail(ctx, MSPCG_EINVAL, "bad argument (1 <= n_inner <= %d)", KMAX);
  if (use_reduced && !ctx->Ls_hat) return fail(ctx, MSPCG_EINVAL, "use_reduced without mspcg_set_reduced_ls");
  cudaStream_t st = (cudaStream_t)stream;
  if (layout == MSPCG_LAYOUT_NATIVE) {
    CUDA_OK(ctx, precond_any(ctx, r_dev, z_dev, io_prec, n_inner, use_reduced != 0, st));
  } else {
    CUDA_OK(ctx, pack_any(ctx, (const double*)r_dev, ctx->stage_in, io_prec, 1, st));
    CUDA_OK(ctx, precond_any(ctx, ctx->stage_in, ctx->stage_out, io_prec, n_inner, use_reduced != 0, st));
    CUDA_OK(ctx, pack_any(ctx, (double*)z_dev, ctx->stage_out, io_prec, 0, st));
  }
  return MSPCG_OK;
}

int mspcg_prepare_source(mspcg_ctx* ctx, const double* phi_e_dev, const double* phi_o_dev, double* phihat_e_dev, double* rhs_dev, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!phi_e_dev || !phi_o_dev || !rhs_dev) return fail(ctx, MSPCG_EINVAL, "null pointer");
  cudaStream_t st = (cudaStream_t)stream;
  double *pe = ctx->v_b, *po = ctx->v_xhi, *hat = ctx->v_rhi, *rhs = ctx->v_t64;
  CUDA_OK(ctx, pack_any(ctx, phi_e_dev, pe, MSPCG_F64, 1, st, 0));
  CUDA_OK(ctx, pack_any(ctx, phi_o_dev, po, MSPCG_F64, 1, st, 1));
  DISPATCH_LS(ctx->Ls, CUDA_OK(ctx, (prepare_source_impl<LS>(ctx, pe, po, hat, rhs, st))));
  if (phihat_e_dev) CUDA_OK(ctx, pack_any(ctx, phihat_e_dev, hat, MSPCG_F64, 0, st, 0));
  CUDA_OK(ctx, pack_any(ctx, rhs_dev, rhs, MSPCG_F64, 0, st, 0));
  return MSPCG_OK;
}
int mspcg_reconstruct_odd(mspcg_ctx* ctx, const double* psi_e_dev, const double* phi_o_dev, double* psi_o_dev, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!psi_e_dev || !phi_o_dev || !psi_o_dev) return fail(ctx, MSPCG_EINVAL, "null pointer");
  cudaStream_t st = (cudaStream_t)stream;
  double *xe = ctx->v_b, *po = ctx->v_xhi, *xo = ctx->v_rhi;
  CUDA_OK(ctx, pack_any(ctx, psi_e_dev, xe, MSPCG_F64, 1, st, 0));
  CUDA_OK(ctx, pack_any(ctx, phi_o_dev, po, MSPCG_F64, 1, st, 1));
  DISPATCH_LS(ctx->Ls, CUDA_OK(ctx, (reconstruct_odd_impl<LS>(ctx, xe, po, xo, st))));
  CUDA_OK(ctx, pack_any(ctx, psi_o_dev, xo, MSPCG_F64, 0, st, 1));
  return MSPCG_OK;
}
int mspcg_apply_full(mspcg_ctx* ctx, const double* psi_e_dev, const double* psi_o_dev, double* out_e_dev, double* out_o_dev, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!psi_e_dev || !psi_o_dev || !out_e_dev || !out_o_dev) return fail(ctx, MSPCG_EINVAL, "null pointer");
  cudaStream_t st = (cudaStream_t)stream;
  double *xe = ctx->v_b, *xo = ctx->v_xhi, *oe = ctx->v_rhi, *oo = ctx->v_t64;
  CUDA_OK(ctx, pack_any(ctx, psi_e_dev, xe, MSPCG_F64, 1, st, 0));
  CUDA_OK(ctx, pack_any(ctx, psi_o_dev, xo, MSPCG_F64, 1, st, 1));
  DISPATCH_LS(ctx->Ls, CUDA_OK(ctx, (apply_full_impl<LS>(ctx, xe, xo, oe, oo, st))));
  CUDA_OK(ctx, pack_any(ctx, out_e_dev, oe, MSPCG_F64, 0, st, 0));
  CUDA_OK(ctx, pack_any(ctx, out_o_dev, oo, MSPCG_F64, 0, st, 1));
  return MSPCG_OK;
}

int mspcg_apply_MdagM_host(mspcg_ctx* ctx, const double* in_host, double* out_host, int prec) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  const size_t n = vec_bytes(ctx, MSPCG_F64, ctx->Ls);
  CUDA_OK(ctx, cudaMemcpyAsync(ctx->abi_in, in_host, n, cudaMemcpyHostToDevice, 0));
  rc = mspcg_apply_MdagM(ctx, ctx->abi_in, ctx->abi_out, prec, MSPCG_LAYOUT_ABI, nullptr); if (rc) return rc;
  CUDA_OK(ctx, cudaMemcpyAsync(out_host, ctx->abi_out, n, cudaMemcpyDeviceToHost, 0));
  CUDA_OK(ctx, cudaStreamSynchronize(0));
  return MSPCG_OK;
}
int mspcg_apply_precond_host(mspcg_ctx* ctx, const double* r_host, double* z_host, int io_prec, int n_inner, int use_reduced) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  const size_t n = vec_bytes(ctx, MSPCG_F64, ctx->Ls);
  CUDA_OK(ctx, cudaMemcpyAsync(ctx->abi_in, r_host, n, cudaMemcpyHostToDevice, 0));
  rc = mspcg_apply_precond(ctx, ctx->abi_in, ctx->abi_out, io_prec, MSPCG_LAYOUT_ABI, n_inner, use_reduced, nullptr); if (rc) return rc;
  CUDA_OK(ctx, cudaMemcpyAsync(z_host, ctx->abi_out, n, cudaMemcpyDeviceToHost, 0));
  CUDA_OK(ctx, cudaStreamSynchronize(0));
  return MSPCG_OK;
}

// The same two calls with SINGLE-precision host vectors (ABI layout, float): for fp32 / fp16 computations the fp64 wire format doubles the
// PCIe bytes of a step that is bound by them.  Device staging: the fp64 ABI buffers, used as float arrays.
int mspcg_apply_MdagM_host32(mspcg_ctx* ctx, const float* in_host, float* out_host, int prec) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!in_host || !out_host || prec == MSPCG_F64 || !full_buf(ctx, prec)) return fail(ctx, MSPCG_EINVAL, "null pointer, or prec is fp64 / not configured (use mspcg_apply_MdagM_host)");
  const size_t n = vec_bytes(ctx, MSPCG_F32, ctx->Ls);
  float *din = (float*)ctx->abi_in, *dout = (float*)ctx->abi_out;
  CUDA_OK(ctx, cudaMemcpyAsync(din, in_host, n, cudaMemcpyHostToDevice, 0));
  CUDA_OK(ctx, pack_any_t<float>(ctx, din, ctx->stage_in, prec, 1, 0, 0));
  CUDA_OK(ctx, normal_full_any(ctx, prec, ctx->stage_in, ctx->stage_out, nullptr, 0));
  CUDA_OK(ctx, pack_any_t<float>(ctx, dout, ctx->stage_out, prec, 0, 0, 0));
  CUDA_OK(ctx, cudaMemcpyAsync(out_host, dout, n, cudaMemcpyDeviceToHost, 0));
  CUDA_OK(ctx, cudaStreamSynchronize(0));
  return MSPCG_OK;
}
int mspcg_apply_precond_host32(mspcg_ctx* ctx, const float* r_host, float* z_host, int io_prec, int n_inner, int use_reduced) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!r_host || !z_host || n_inner < 1 || n_inner > KMAX || (io_prec != MSPCG_F32 && io_prec != MSPCG_F16)) return fail(ctx, MSPCG_EINVAL, "bad argument (io_prec fp32 or fp16, 1 <= n_inner <= %d)", KMAX);
  if (use_reduced && !ctx->Ls_hat) return fail(ctx, MSPCG_EINVAL, "use_reduced without mspcg_set_reduced_ls");
  const size_t n = vec_bytes(ctx, MSPCG_F32, ctx->Ls);
  float *din = (float*)ctx->abi_in, *dout = (float*)ctx->abi_out;
  CUDA_OK(ctx, cudaMemcpyAsync(din, r_host, n, cudaMemcpyHostToDevice, 0));
  CUDA_OK(ctx, pack_any_t<float>(ctx, din, ctx->stage_in, io_prec, 1, 0, 0));
  CUDA_OK(ctx, precond_any(ctx, ctx->stage_in, ctx->stage_out, io_prec, n_inner, use_reduced != 0, 0));
  CUDA_OK(ctx, pack_any_t<float>(ctx, dout, ctx->stage_out, io_prec, 0, 0, 0));
  CUDA_OK(ctx, cudaMemcpyAsync(z_host, dout, n, cudaMemcpyDeviceToHost, 0));
  CUDA_OK(ctx, cudaStreamSynchronize(0));
  return MSPCG_OK;
}

int mspcg_apply_A_block(mspcg_ctx* ctx, const double* in_dev, double* out_dev, int block, int prec, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!in_dev || !out_dev || block < 0 || block >= ctx->lat.nblk || prec != ctx->inner_prec) return fail(ctx, MSPCG_EINVAL, "bad argument (prec must be the configured inner_prec)");
  cudaStream_t st = (cudaStream_t)stream;
  const Geometry& g = ctx->lat.blk;
  const size_t blk_bytes = (size_t)g.nE0 * ctx->Ls * 24 * prec;
  CUDA_OK(ctx, pack_any(ctx, in_dev, ctx->stage_in, prec, 1, st));
  CUDA_OK(ctx, cudaMemsetAsync(ctx->stage_out, 0, vec_bytes(ctx, prec, ctx->Ls), st));
  const char* pin = (const char*)ctx->stage_in + blk_bytes * block;
  char* pout = (char*)ctx->stage_out + blk_bytes * block;
  ctx->cur_geom = 1;
#define AB(TT) { OpView<TT> v = one_block(make_view<TT>(ctx, ctx->blkI, g, ctx->gblk, ctx->Ls, false), block); \
    DISPATCH_LS(ctx->Ls, CUDA_OK(ctx, (apply_normal<TT, LS>(ctx, v, mphi_plain<TT>((const TT*)pin), (const TT*)pin, (TT*)pout, nullptr, st)))); }
  if (prec == MSPCG_F64) AB(double) else if (prec == MSPCG_F32) AB(float) else AB(__half)
#undef AB
  CUDA_OK(ctx, pack_any(ctx, out_dev, ctx->stage_out, prec, 0, st));
  return MSPCG_OK;
}

int mspcg_solve(mspcg_ctx* ctx, const double* b_dev, double* x_dev, const mspcg_solve_params* params,
                mspcg_solve_stats* stats, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!b_dev || !x_dev || !params || !stats) return fail(ctx, MSPCG_EINVAL, "null argument");
  if (params->use_precond && (params->n_inner < 1 || params->n_inner > KMAX)) return fail(ctx, MSPCG_EINVAL, "bad n_inner");
  if (params->use_reduced_ls && !(params->use_precond && ctx->Ls_hat)) return fail(ctx, MSPCG_EINVAL, "use_reduced_ls needs use_precond and mspcg_set_reduced_ls");
  if (!full_buf(ctx, params->sloppy_prec)) return fail(ctx, MSPCG_EINVAL, "sloppy_prec not configured");
  cudaStream_t st = (cudaStream_t)stream;
  if (params->sloppy_prec == MSPCG_F64) return solve_impl<double>(ctx, b_dev, x_dev, params, stats, st);
  if (params->sloppy_prec == MSPCG_F32) return solve_impl<float>(ctx, b_dev, x_dev, params, stats, st);
  return solve_impl<__half>(ctx, b_dev, x_dev, params, stats, st);
}

int mspcg_residual(mspcg_ctx* ctx, const double* b_dev, const double* x_dev, double* r_dev, int normalise, double* rnorm_host, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!b_dev || !x_dev || !r_dev || r_dev == b_dev || r_dev == x_dev) return fail(ctx, MSPCG_EINVAL, "null pointer or aliasing");
  cudaStream_t st = (cudaStream_t)stream;
  const long nreal = v5h(ctx, ctx->Ls) * 24;
  double *b = ctx->v_b, *x = ctx->v_xhi, *r = ctx->v_rhi, *t = ctx->v_t64;
  CUDA_OK(ctx, pack_any(ctx, b_dev, b, MSPCG_F64, 1, st));
  CUDA_OK(ctx, pack_any(ctx, x_dev, x, MSPCG_F64, 1, st));
  CUDA_OK(ctx, normal_full<double>(ctx, ctx->full64, x, t, mphi_plain<double>(x), nullptr, st));
  CUDA_OK(ctx, cudaMemcpyAsync(r, b, sizeof(double) * nreal, cudaMemcpyDeviceToDevice, st));
  CUDA_OK(ctx, axpby<double>(ctx, -1.0, t, 1.0, r, nreal, st));
  CUDA_OK(ctx, cudaMemsetAsync(ctx->sc + 8, 0, sizeof(double), st));
  CUDA_OK(ctx, dot2<double>(ctx, r, r, nullptr, nreal, st, ctx->sc + 8));
  CUDA_OK(ctx, sc_read(ctx, 16, st));
  const double rn = std::sqrt(ctx->sc_host[8]);
  if (rnorm_host) *rnorm_host = rn;
  if (normalise && rn > 0.0) CUDA_OK(ctx, axpby<double>(ctx, 0.0, r, 1.0 / rn, r, nreal, st));
  CUDA_OK(ctx, pack_any(ctx, r_dev, r, MSPCG_F64, 0, st));
  CUDA_OK(ctx, cudaStreamSynchronize(st));
  return MSPCG_OK;
}

int mspcg_update_T(mspcg_ctx* ctx, const double* T_host, double mu, void* stream) {
  int rc = check_ready(ctx, false); if (rc) return rc;
  if (!ctx->Ls_hat || !T_host) return fail(ctx, MSPCG_EINVAL, "mspcg_update_T needs mspcg_set_reduced_ls before the workspace was sized");
  ctx->T_host.assign(T_host, T_host + (size_t)4 * ctx->Ls_hat * 4 * ctx->Ls * 2);
  ctx->mu_shift = mu;
  return upload_T(ctx, (cudaStream_t)stream);
}

int mspcg_train_eval(mspcg_ctx* ctx, const double* v_dev, int nvec, int n_inner, double* chi2_host, double* grad_host, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!ctx->Ls_hat || !v_dev || nvec < 1 || !chi2_host || n_inner < 1 || n_inner > KMAX) return fail(ctx, MSPCG_EINVAL, "bad argument or no reduced-Ls set-up");
  if (ctx->inner_prec == MSPCG_F16) return fail(ctx, MSPCG_EINVAL, "training runs with inner_prec fp64 or fp32 (train there, use T anywhere)");
  mspcg_ctx* c = ctx;
  if (ctx->inner_prec == MSPCG_F64) return train_eval_impl<double>(c, v_dev, nvec, n_inner, chi2_host, grad_host, (cudaStream_t)stream);
  return train_eval_impl<float>(c, v_dev, nvec, n_inner, chi2_host, grad_host, (cudaStream_t)stream);
}

int mspcg_train_T(mspcg_ctx* ctx, const double* v_dev, int nvec, int n_inner, int n_steps, double momentum, double* T_host_out,
                  double* chi2_history_host, void* stream) {
  int rc = check_ready(ctx, true); if (rc) return rc;
  if (!ctx->Ls_hat || n_steps < 0 || !T_host_out) return fail(ctx, MSPCG_EINVAL, "bad argument or no reduced-Ls set-up");
  const size_t n = (size_t)16 * ctx->Ls_hat * ctx->Ls * 2;
  std::vector<double> T(ctx->T_host), G(n), P(n, 0.0), Tt(n);
  const double mu = ctx->mu_shift;
  double val = 0, scale = 1.0;
  for (int step = 0; step < n_steps; step++) {
    if ((rc = mspcg_train_eval(ctx, v_dev, nvec, n_inner, &val, G.data(), stream))) return rc;
    if (chi2_history_host) chi2_history_host[step] = val;
    double g2 = 0; for (size_t i = 0; i < n; i++) g2 += G[i] * G[i];
    if (!(g2 > 0)) break;
    for (size_t i = 0; i < n; i++) P[i] = -G[i] + momentum * P[i];                // momentum method ([25])
    const double eta0 = scale * val / g2;
    const double eta[5] = {0.0, 0.5 * eta0, eta0, 1.5 * eta0, 2.0 * eta0};
    double vals[5] = {val, 0, 0, 0, 0};
    for (int j = 1; j < 5; j++) {
      for (size_t i = 0; i < n; i++) Tt[i] = T[i] + eta[j] * P[i];
      if ((rc = mspcg_update_T(ctx, Tt.data(), mu, stream))) return rc;
      if ((rc = mspcg_train_eval(ctx, v_dev, nvec, n_inner, &vals[j], nullptr, stream))) return rc;
    }
    double es = quartic_argmin(eta, vals);
    int best = 0; for (int j = 1; j < 5; j++) if (vals[j] < vals[best]) best = j;
    bool sampled = false; for (int j = 0; j < 5; j++) sampled = sampled || es == eta[j];
    if (!sampled) {   // the fit promised more than the loss delivers: keep the best measured point
      double ve = 0;
      for (size_t i = 0; i < n; i++) Tt[i] = T[i] + es * P[i];
      if ((rc = mspcg_update_T(ctx, Tt.data(), mu, stream))) return rc;
      if ((rc = mspcg_train_eval(ctx, v_dev, nvec, n_inner, &ve, nullptr, stream))) return rc;
      if (ve > vals[best]) es = eta[best];
    }
    for (size_t i = 0; i < n; i++) T[i] += es * P[i];
    if (es == 0.0) { std::fill(P.begin(), P.end(), 0.0); scale *= 0.25; }   // no decrease found: drop the momentum, shorten the step
    else scale = std::fmin(1.0, scale * 2.0);
    if ((rc = mspcg_update_T(ctx, T.data(), mu, stream))) return rc;
  }
  if ((rc = mspcg_train_eval(ctx, v_dev, nvec, n_inner, &val, nullptr, stream))) return rc;
  if (chi2_history_host) chi2_history_host[n_steps] = val;
  memcpy(T_host_out, T.data(), n * sizeof(double));
  return MSPCG_OK;
}

int mspcg_tile_check(mspcg_ctx* ctx, double out_host[8]) {
  if (!ctx || !out_host) return MSPCG_EINVAL;
  TileSet tb, tf;
  build_tile_set(tb, ctx->lat.blk); build_tile_set(tf, ctx->lat.full);
  const Geometry &g = ctx->lat.blk, &f = ctx->lat.full;
  int bad = 0, code;
  if ((code = check_tiles(tb.hO_lim, g.nbrO, 0, g.nO, g.nE0))) bad = 100 + code;
  else if (!tb.hO_all.empty() && (code = check_tiles(tb.hO_all, g.nbrO, 0, g.nO, g.nE))) bad = 200 + code;
  else if ((code = check_tiles(tb.hE_int, g.nbrE, 0, g.nE0, g.nO))) bad = 300 + code;
  else if ((code = check_tiles(tb.hE_halo, g.nbrE, g.nE0, g.nE, g.nO))) bad = 400 + code;
  else if ((code = check_tiles(tf.hO_lim, f.nbrO, 0, f.nO, f.nE0))) bad = 500 + code;
  else if ((code = check_tiles(tf.hE_int, f.nbrE, 0, f.nE0, f.nO))) bad = 600 + code;
  const std::vector<TileRec>& k4 = tb.hO_all.empty() ? tb.hO_lim : tb.hO_all;
  out_host[0] = bad;
  out_host[1] = (double)tb.hO_lim.size(); out_host[2] = (double)k4.size(); out_host[3] = (double)tb.hE_int.size(); out_host[4] = (double)tb.hE_halo.size();
  out_host[5] = tiles_inputs_per_output(k4); out_host[6] = tiles_inputs_per_output(tb.hE_int); out_host[7] = tiles_inputs_per_output(tf.hE_int);
  return bad ? fail(ctx, MSPCG_EINVAL, "tile tables inconsistent with the neighbour tables (code %d)", bad) : MSPCG_OK;
}

int mspcg_set_block_group(mspcg_ctx* ctx, int blocks_per_group) {
  if (!ctx || blocks_per_group < 0) return MSPCG_EINVAL;
  ctx->group_blocks = blocks_per_group;
  return MSPCG_OK;
}

int mspcg_set_fixed_storage(mspcg_ctx* ctx, int bits) {
  if (!ctx) return MSPCG_EINVAL;
  if (bits != 0 && bits != 8 && bits != 16) return fail(ctx, MSPCG_EINVAL, "mspcg_set_fixed_storage: bits must be 0, 8 or 16");
  ctx->fixed_bits = bits;
  return MSPCG_OK;
}

int mspcg_fixed_pack(mspcg_ctx* ctx, const double* abi_dev, void* q_dev, float* scale_dev, int bits, void* stream) {
  if (!ctx) return MSPCG_EINVAL;
  if (!abi_dev || !q_dev || !scale_dev || (bits != 8 && bits != 16)) return fail(ctx, MSPCG_EINVAL, "mspcg_fixed_pack: null pointer or bits not 8 / 16");
  const long ncs = v5h(ctx, ctx->Ls);
  const unsigned grid = (unsigned)((ncs + 127) / 128);
  if (bits == 8) k_fixed_pack<int8_t><<<grid, 128, 0, (cudaStream_t)stream>>>(abi_dev, (int8_t*)q_dev, scale_dev, ncs);
  else k_fixed_pack<int16_t><<<grid, 128, 0, (cudaStream_t)stream>>>(abi_dev, (int16_t*)q_dev, scale_dev, ncs);
  ctx->launches++;
  CUDA_OK(ctx, cudaPeekAtLastError());
  return MSPCG_OK;
}

int mspcg_fixed_unpack(mspcg_ctx* ctx, const void* q_dev, const float* scale_dev, double* abi_dev, int bits, void* stream) {
  if (!ctx) return MSPCG_EINVAL;
  if (!abi_dev || !q_dev || !scale_dev || (bits != 8 && bits != 16)) return fail(ctx, MSPCG_EINVAL, "mspcg_fixed_unpack: null pointer or bits not 8 / 16");
  const long ncs = v5h(ctx, ctx->Ls);
  const unsigned grid = (unsigned)((ncs + 127) / 128);
  if (bits == 8) k_fixed_unpack<int8_t><<<grid, 128, 0, (cudaStream_t)stream>>>((const int8_t*)q_dev, scale_dev, abi_dev, ncs);
  else k_fixed_unpack<int16_t><<<grid, 128, 0, (cudaStream_t)stream>>>((const int16_t*)q_dev, scale_dev, abi_dev, ncs);
  ctx->launches++;
  CUDA_OK(ctx, cudaPeekAtLastError());
  return MSPCG_OK;
}

long mspcg_launch_count(const mspcg_ctx* ctx) { return ctx ? ctx->launches : 0; }

int mspcg_timing(mspcg_ctx* ctx, int enable) {
  if (!ctx) return MSPCG_EINVAL;
  ctx->timing = enable != 0; ctx->ev_used = 0; ctx->ev_cls.clear();
  return MSPCG_OK;
}

int mspcg_timing_read(mspcg_ctx* ctx, double* ms_host, long* launches_host) {
  if (!ctx || !ms_host || !launches_host) return MSPCG_EINVAL;
  for (int i = 0; i < NCLASS; i++) { ms_host[i] = 0; launches_host[i] = 0; }
  CUDA_OK(ctx, cudaDeviceSynchronize());
  for (size_t i = 0; i < ctx->ev_cls.size(); i++) {
    float ms = 0;
    CUDA_OK(ctx, cudaEventElapsedTime(&ms, ctx->ev_pool[2 * i], ctx->ev_pool[2 * i + 1]));
    ms_host[ctx->ev_cls[i]] += ms; launches_host[ctx->ev_cls[i]]++;
  }
  ctx->ev_used = 0; ctx->ev_cls.clear();
  return MSPCG_OK;
}

}  // extern "C"

// ======================================================================================================================
// mspcg_dot2_noalloc: the two inner products of the Polak-Ribiere beta (eq. 18, R16; k_dot2 in kernels.cuh) for callers
// that cannot allocate (CUDA graph capture, serving loops): no context, no workspace.  k_dot2 accumulates with atomics into
// scratch scalars of the caller's workspace; this variant keeps its scratch -- one pair of partial sums per CHUNK of the
// vectors and a ticket counter -- in the file-scope device array below, which every GPU that loads the library holds until
// exit (NOALLOC_BYTES = 513 KiB).  The result does not depend on the grid size or on the order in which thread blocks finish.
// ======================================================================================================================
namespace {

constexpr long NOALLOC_CHUNK = 16384;                 // reals per partial sum (one thread block pass)
constexpr long NOALLOC_MAX_CHUNKS = 32768;            // => at most 2^29 reals (4 GiB of fp64) per vector
constexpr long NOALLOC_MAX_REALS = NOALLOC_CHUNK * NOALLOC_MAX_CHUNKS;
constexpr size_t NOALLOC_BYTES = sizeof(double) * 2 * NOALLOC_MAX_CHUNKS + 256;   // partial sums, then the ticket counter
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

// grid-stride over chunks; partial[2 c], partial[2 c + 1] = <a,b>, <a,c> over chunk c, summed in a fixed order; the thread block
// that draws the last ticket adds the partial sums in a fixed order and writes out[0..1].
__global__ void __launch_bounds__(256) k_dot2_static(const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ c,
                                                     long n, long nchunks, double* partial, unsigned int* ticket, double* out) {
  __shared__ double red[32];
  __shared__ bool last;
  for (long ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
    const long lo = ch * NOALLOC_CHUNK, hi = lo + NOALLOC_CHUNK < n ? lo + NOALLOC_CHUNK : n;
    double p0 = 0, p1 = 0;
    for (long i = lo + threadIdx.x; i < hi; i += 256) {
      const double va = a[i];
      p0 += va * b[i];
      if (c) p1 += va * c[i];
    }
    const double t0 = block_sum(p0, red, threadIdx.x, 256);
    __syncthreads();
    const double t1 = block_sum(p1, red, threadIdx.x, 256);
    __syncthreads();
    if (threadIdx.x == 0) { partial[2 * ch] = t0; partial[2 * ch + 1] = t1; }
  }
  if (threadIdx.x == 0) {
    __threadfence();
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double s0 = 0, s1 = 0;
  for (long ch = threadIdx.x; ch < nchunks; ch += 256) { s0 += __ldcg(partial + 2 * ch); s1 += __ldcg(partial + 2 * ch + 1); }
  const double t0 = block_sum(s0, red, threadIdx.x, 256);
  __syncthreads();
  const double t1 = block_sum(s1, red, threadIdx.x, 256);
  if (threadIdx.x == 0) { out[0] = t0; out[1] = t1; *ticket = 0; }
}

std::mutex g_noalloc_mu;
unsigned char* g_noalloc_ptr[NOALLOC_MAX_DEVICES];    // device address of g_noalloc_scratch on each device (host code cannot use the symbol's name as a pointer)
int g_noalloc_sms[NOALLOC_MAX_DEVICES];
thread_local char g_noalloc_err[256] = "";

int noalloc_fail(int code, const char* fmt, ...) {
  va_list ap; va_start(ap, fmt); vsnprintf(g_noalloc_err, sizeof(g_noalloc_err), fmt, ap); va_end(ap);
  return code;
}

}  // namespace

extern "C" {

const char* mspcg_noalloc_last_error(void) { return g_noalloc_err; }
long mspcg_dot2_noalloc_max_reals(void) { return NOALLOC_MAX_REALS; }

int mspcg_dot2_noalloc(const double* a_dev, const double* b_dev, const double* c_dev, long n_reals, double* out_dev, void* stream) {
  if (!out_dev || (n_reals > 0 && (!a_dev || !b_dev))) return noalloc_fail(MSPCG_EINVAL, "mspcg_dot2_noalloc: null pointer");
  if (n_reals < 0 || n_reals > NOALLOC_MAX_REALS)
    return noalloc_fail(MSPCG_EINVAL, "mspcg_dot2_noalloc: n_reals = %ld is outside [0, %ld] (the static scratch holds %ld partial sums of %ld reals)",
                        n_reals, NOALLOC_MAX_REALS, NOALLOC_MAX_CHUNKS, NOALLOC_CHUNK);
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return noalloc_fail(MSPCG_ECUDA, "mspcg_dot2_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return noalloc_fail(MSPCG_EINVAL, "mspcg_dot2_noalloc: device ordinal %d >= %d", dev, NOALLOC_MAX_DEVICES);
  unsigned char* base; int sms;
  {   // once per device, with that device current: the device address of the scratch array
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
      if (e != cudaSuccess || !p) return noalloc_fail(MSPCG_ECUDA, "mspcg_dot2_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
      int n = 0;
      e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
      if (e != cudaSuccess || n < 1) return noalloc_fail(MSPCG_ECUDA, "mspcg_dot2_noalloc: cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
      g_noalloc_sms[dev] = n;
      g_noalloc_ptr[dev] = (unsigned char*)p;
    }
    base = g_noalloc_ptr[dev]; sms = g_noalloc_sms[dev];
  }
  cudaStream_t st = (cudaStream_t)stream;
  double* partial = reinterpret_cast<double*>(base);
  unsigned int* ticket = reinterpret_cast<unsigned int*>(base + sizeof(double) * 2 * NOALLOC_MAX_CHUNKS);
  // the array keeps the last call's contents: the ticket must start at zero (the partial sums are overwritten before they are read)
  e = cudaMemsetAsync(ticket, 0, sizeof(unsigned int), st);
  if (e != cudaSuccess) return noalloc_fail(MSPCG_ECUDA, "mspcg_dot2_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
  const long nchunks = (n_reals + NOALLOC_CHUNK - 1) / NOALLOC_CHUNK;
  const long want = nchunks < 1 ? 1 : nchunks, cap = 8L * sms;
  k_dot2_static<<<(unsigned)(want < cap ? want : cap), 256, 0, st>>>(a_dev, b_dev, c_dev, n_reals, nchunks, partial, ticket, out_dev);
  e = cudaPeekAtLastError();
  if (e != cudaSuccess) return noalloc_fail(MSPCG_ECUDA, "mspcg_dot2_noalloc: launch: %s", cudaGetErrorString(e));
  return MSPCG_OK;
}

}  // extern "C"
