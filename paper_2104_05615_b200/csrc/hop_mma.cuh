// hop_mma.cuh -- the fused hop kernel for fp16 storage (the preconditioner's hot path): one WARP
// owns one 4D site and its whole fifth-dimension column; the SU(3) x half-spinor products and the Ls x Ls fifth-dimension
// contractions both run on the tensor cores with fp16 operands and fp32 accumulation; the CUDA cores do the spin
// projection (packed fp16 adds), the reconstruction of the lower components (32 FMAs per site column) and conversions.
//
// fp16 vector layout in HBM (private NATIVE layout of the __half storage type, see ST<__half> in kernels.cuh):
//     v[site][s][colour t (3)][sp (2)][hi (2)][re,im]          spin = 2*hi + sp   (hi = 0: P+ rows, hi = 1: P- rows)
// i.e. 48 contiguous bytes per (site, s), three 16-byte chunks, one per colour.  Lane (g = lane/4, t = lane%4) of the
// warp reads the chunk {u0, l0, u1, l1} of colour t for s = g and s = 8 + g (u = upper, l = lower two-spinor).
//
//   hop (eq. 8), per direction:  (1 + c gamma_mu) W psi,  c = -sg (forward), +sg (backward), W the link.
//       In the chiral basis (reading R2) its upper part is W h with the half spinor h = u + c G l (G = -i sigma_k, 1 for
//       mu = t) and its lower part is c G^dag (W h).  h is formed in the lane with packed fp16 FMAs and is the A fragment
//       of mma.m16n8k16: rows (sp, s mod 8), one M-tile per segment of eight s, K = forward colours | backward colours
//       (lanes t = 3 pad K with zeros).  The B fragment is the link as a real 6x6 (padded 8x8) matrix, built from one
//       32-bit load per lane.  One MMA accumulates the upper components over all directions; a second one with the
//       forward half of B negated gives W_b h_b - W_f h_f, which sg G^dag maps onto the lower components inside the lane.
//   5D matrices: out[s][n] = sum_s' M_hi[s][s'] X[s'][n]; the accumulator fragment is
//       converted to fp16 (the paper's HMMA operands), transposed across the warp with movmatrix into a
//       B fragment, and multiplied by the constant A fragment of M (host-built, one uint4 per lane and chirality).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace mspcg {

template <int LS> struct MmaCfg {
  enum { NSEG = LS > 8 ? 2 : 1, N0 = LS > 8 ? 8 : LS, N1 = LS > 8 ? LS - 8 : 0, NMT = 2 * NSEG, NW = 4 };
};

__device__ __forceinline__ void mma16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t x) {
  uint32_t y;
  asm("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;\n" : "=r"(y) : "r"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack_h2(float lo, float hi) {
  __half2 h = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ float2 unpack_h2(uint32_t u) { return __half22float2(*reinterpret_cast<__half2*>(&u)); }

// Fragment of the vector at `site`: f[seg] = 16-byte chunk of colour t at s = 8*seg + g (zero where the lane pads).
template <int LS>
__device__ __forceinline__ void load_frag(const __half* __restrict__ base, long site, int g, int t, uint4 (&f)[MmaCfg<LS>::NSEG], bool ok = true) {
  typedef MmaCfg<LS> Cfg;
  const uint4* p = reinterpret_cast<const uint4*>(base) + (ok ? site : 0) * (LS * 3) + g * 3 + t;
  f[0] = (ok && t < 3 && g < Cfg::N0) ? __ldg(p) : make_uint4(0, 0, 0, 0);
  if (Cfg::NSEG == 2) f[Cfg::NSEG - 1] = (ok && t < 3 && g < Cfg::N1) ? __ldg(p + 24) : make_uint4(0, 0, 0, 0);
}
template <int LS>
__device__ __forceinline__ void store_frag(__half* __restrict__ base, long site, int g, int t, const uint4 (&f)[MmaCfg<LS>::NSEG]) {
  typedef MmaCfg<LS> Cfg;
  uint4* p = reinterpret_cast<uint4*>(base) + site * (LS * 3) + g * 3 + t;
  if (t < 3 && g < Cfg::N0) p[0] = f[0];
  if (Cfg::NSEG == 2) { if (t < 3 && g < Cfg::N1) p[24] = f[Cfg::NSEG - 1]; }
}

// B fragment of one link from its raw word.  Raw word of lane (g, t): the complex half2 W[c = g/2][t] of the stored
// link (NG = 18: nine complex halves row-major; NG = 12: rows 0 and 1 only, reading R8), zero on pad lanes.
// Lane (g, t) supplies B[k = (colour t, re/im)][n = g = (row colour c, re/im = g%2)]: (Wr, -Wi) for the real output
// column, (Wi, Wr) for the imaginary one -- one byte permute with the per-lane selector `sel` (0x7610 / 0x1032).
// With NG = 12 the lanes of row 2 get conj(row0 x row1) from the lanes holding rows 0 and 1 (lane t' holds a_t',
// lane 8 + t' holds b_t'); executed by the whole warp (shuffles).
template <int NG>
__device__ __forceinline__ uint32_t link_bfrag(uint32_t raw, int g, int t, uint32_t sel) {
  uint32_t w = raw;
  if (NG == 12) {
    const int tt = t == 3 ? 0 : t;
    const int t1 = tt == 2 ? 0 : tt + 1, t2 = tt == 0 ? 2 : tt - 1;   // (t+1)%3, (t+2)%3
    const float2 a1 = unpack_h2(__shfl_sync(0xffffffffu, raw, t1)), b2 = unpack_h2(__shfl_sync(0xffffffffu, raw, 8 + t2));
    const float2 a2 = unpack_h2(__shfl_sync(0xffffffffu, raw, t2)), b1 = unpack_h2(__shfl_sync(0xffffffffu, raw, 8 + t1));
    const float re = (a1.x * b2.x - a1.y * b2.y) - (a2.x * b1.x - a2.y * b1.y);
    const float im = (a1.x * b2.y + a1.y * b2.x) - (a2.x * b1.y + a2.y * b1.x);
    if ((g >> 1) == 2 && t < 3) w = pack_h2(re, -im);
  }
  return __byte_perm(w, w ^ 0x80000000u, sel);   // pad lanes: (+0, -0), harmless
}

// Half-spinor projection BEFORE the SU(3) product.  (1 + c gamma_mu) psi has upper part
// h = u + c G l and lower part c G^dag h  (G = -i sigma_k, or 1 for mu = t; c = -sg forward, +sg backward), so only h (two spin
// components) is multiplied by the link: rows of the MMA are (sp, s) and one M-tile covers a whole segment, i.e. half the MMAs
// and half the fragment reads of a full-spinor product.  h is rounded to fp16, the MMA operand precision.
__device__ __forceinline__ uint32_t hfma2_u32(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t d;
  asm("fma.rn.f16x2 %0, %1, %2, %3;\n" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}
__device__ __forceinline__ uint32_t swap_h2(uint32_t x) { return __byte_perm(x, x, 0x1032); }
struct HsConst { uint32_t P, N, Q, R; };   // half2 (sg,sg), (-sg,-sg), (sg,-sg), (-sg,sg)
// chunk = {u0, l0, u1, l1} (half2 re,im each); fwd: c = -sg, bwd: c = +sg
template <int MU, bool FWD>
__device__ __forceinline__ void project_hs(const uint4& q, const HsConst& k, uint32_t& h0, uint32_t& h1) {
  if (MU == 0)      { const uint32_t m = FWD ? k.R : k.Q; h0 = hfma2_u32(swap_h2(q.w), m, q.x); h1 = hfma2_u32(swap_h2(q.y), m, q.z); }
  else if (MU == 1) { h0 = hfma2_u32(q.w, FWD ? k.P : k.N, q.x); h1 = hfma2_u32(q.y, FWD ? k.N : k.P, q.z); }
  else if (MU == 2) { h0 = hfma2_u32(swap_h2(q.y), FWD ? k.R : k.Q, q.x); h1 = hfma2_u32(swap_h2(q.w), FWD ? k.Q : k.R, q.z); }
  else              { const uint32_t m = FWD ? k.N : k.P; h0 = hfma2_u32(q.y, m, q.x); h1 = hfma2_u32(q.w, m, q.z); }
}
__device__ __forceinline__ void mma16816_4(float& d0, float& d1, float& d2, float& d3, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
      : "+f"(d0), "+f"(d1), "+f"(d2), "+f"(d3) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// S[2*seg + sp][hi*2 + ri]: hi = 0 accumulates W h directly; hi = 1 gets sg G^dag (W_b h_b - W_f h_f).
template <int MU, int LS>
__device__ __forceinline__ void hop_mu_hs(float (&S)[MmaCfg<LS>::NMT][4], const uint4 (&F)[MmaCfg<LS>::NSEG], const uint4 (&B)[MmaCfg<LS>::NSEG],
                                          uint32_t bf, uint32_t bb, float sg, const HsConst& k) {
  typedef MmaCfg<LS> Cfg;
  const uint32_t bfn = bf ^ 0x80008000u;
#pragma unroll
  for (int seg = 0; seg < Cfg::NSEG; seg++) {
    uint32_t f0, f1, b0, b1;
    project_hs<MU, true>(F[seg], k, f0, f1);
    project_hs<MU, false>(B[seg], k, b0, b1);
    float (&S0)[4] = S[2 * seg], (&S1)[4] = S[2 * seg + 1];
    mma16816_4(S0[0], S0[1], S1[0], S1[1], f0, f1, b0, b1, bf, bb);
    float d0 = 0.f, d1 = 0.f, d2 = 0.f, d3 = 0.f;   // (sp0 re, im), (sp1 re, im) of W_b h_b - W_f h_f
    mma16816_4(d0, d1, d2, d3, f0, f1, b0, b1, bfn, bb);
    if (MU == 0)      { S0[2] -= sg * d3; S0[3] += sg * d2; S1[2] -= sg * d1; S1[3] += sg * d0; }   // i sigma_1
    else if (MU == 1) { S0[2] += sg * d2; S0[3] += sg * d3; S1[2] -= sg * d0; S1[3] -= sg * d1; }   // i sigma_2 = [[0,1],[-1,0]]
    else if (MU == 2) { S0[2] -= sg * d1; S0[3] += sg * d0; S1[2] += sg * d3; S1[3] -= sg * d2; }   // i sigma_3 = diag(i,-i)
    else              { S0[2] += sg * d0; S0[3] += sg * d1; S1[2] += sg * d2; S1[3] += sg * d3; }
  }
}
__device__ __forceinline__ uint4 lds128v(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];\n" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}

// X <- M X over the fifth dimension (both chiralities): X is the accumulator fragment set [seg*2+sp][hi*2+ri];
// mfrag[hi*32 + lane] is the A fragment of the 16x16 zero-padded matrix of chirality hi (shared-memory copy).
template <int LS>
__device__ __forceinline__ void dense5d_mma(float (&X)[MmaCfg<LS>::NMT][4], const uint4* __restrict__ mfrag, int lane) {
  typedef MmaCfg<LS> Cfg;
#pragma unroll
  for (int hi = 0; hi < 2; hi++) {
    const uint4 A = mfrag[hi * 32 + lane];
#pragma unroll
    for (int sp = 0; sp < 2; sp++) {
      const uint32_t b0 = movmatrix_trans(pack_h2(X[sp][2 * hi], X[sp][2 * hi + 1]));
      uint32_t b1 = 0u;
      if (Cfg::NSEG == 2) b1 = movmatrix_trans(pack_h2(X[Cfg::NMT - 2 + sp][2 * hi], X[Cfg::NMT - 2 + sp][2 * hi + 1]));
      float d[4] = {0.f, 0.f, 0.f, 0.f};
      mma16816(d, A.x, A.y, A.z, A.w, b0, b1);
      X[sp][2 * hi] = d[0]; X[sp][2 * hi + 1] = d[1];
      if (Cfg::NSEG == 2) { X[Cfg::NMT - 2 + sp][2 * hi] = d[2]; X[Cfg::NMT - 2 + sp][2 * hi + 1] = d[3]; }
    }
  }
}

template <int LS>
__device__ __forceinline__ void frag_to_float(const uint4 (&f)[MmaCfg<LS>::NSEG], float (&X)[MmaCfg<LS>::NMT][4]) {
#pragma unroll
  for (int seg = 0; seg < MmaCfg<LS>::NSEG; seg++) {
    float2 q;
    q = unpack_h2(f[seg].x); X[2 * seg][0] = q.x; X[2 * seg][1] = q.y;
    q = unpack_h2(f[seg].y); X[2 * seg][2] = q.x; X[2 * seg][3] = q.y;
    q = unpack_h2(f[seg].z); X[2 * seg + 1][0] = q.x; X[2 * seg + 1][1] = q.y;
    q = unpack_h2(f[seg].w); X[2 * seg + 1][2] = q.x; X[2 * seg + 1][3] = q.y;
  }
}
template <int LS>
__device__ __forceinline__ void float_to_frag(const float (&X)[MmaCfg<LS>::NMT][4], uint4 (&f)[MmaCfg<LS>::NSEG]) {
#pragma unroll
  for (int seg = 0; seg < MmaCfg<LS>::NSEG; seg++) {
    f[seg].x = pack_h2(X[2 * seg][0], X[2 * seg][1]); f[seg].y = pack_h2(X[2 * seg][2], X[2 * seg][3]);
    f[seg].z = pack_h2(X[2 * seg + 1][0], X[2 * seg + 1][1]); f[seg].w = pack_h2(X[2 * seg + 1][2], X[2 * seg + 1][3]);
  }
}

// ---- per-warp TMA staging (cp.async.bulk, mbarrier) ------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

template <int LS> struct MmaSmem {
  enum { SLOT = LS * 48, STAGE = 8 * SLOT, WARP = 2 * STAGE + 64, BLOCK = MmaCfg<LS>::NW * WARP };   // bytes
};

// The fused hop kernel, fp16 storage.  Same arguments and epilogues as k_hop (kernels.cuh); a.frag1 / a.frag2 are the
// A fragments of the fifth-dimension matrices.  Persistent warps: grid = (gx, nblk), block = 32 * NW threads; warp w of
// the gx*NW warps of a block row takes sites w, w + gx*NW, ...   Every warp runs its own two-stage pipeline:
//   * the eight neighbour columns of a site (Ls*48 contiguous bytes each) are fetched by eight cp.async.bulk copies
//     (one per lane 0..7) into the warp's shared-memory stage and signalled on the warp's mbarrier; the copies of
//     site i+1 are issued before site i is computed, so a full site is always in flight per warp;
//   * neighbour tables, link words, boundary-flip byte and the xpay operand are register-prefetched two sites ahead
//     in two ping-pong register sets (no register is copied, so no step waits for a load it has just issued);
//   * the neighbour chunks are 128-bit shared-memory reads (conflict-free: a quarter warp reads 112 contiguous bytes).
// Slots of absent neighbours (Dirichlet cut) keep stale finite data and meet a zero B fragment.
template <int LS, int EPI, int NG>
__global__ void __launch_bounds__(32 * MmaCfg<LS>::NW, 4) k_hop_mma(const HopArgs<__half> a) {
  typedef MmaCfg<LS> Cfg;
  typedef MmaSmem<LS> SM;
  constexpr int NSEG = Cfg::NSEG, NMT = Cfg::NMT, NW = Cfg::NW;
  extern __shared__ __align__(128) unsigned char smraw[];
  __shared__ double red[NW];
  __shared__ uint4 sfrag[(EPI == EPI_K3 ? 2 : 1) * 64];   // A fragments of the 5D matrices, fetched once per thread block
  if (threadIdx.x < 64) sfrag[threadIdx.x] = __ldg(a.frag1 + threadIdx.x);
  if (EPI == EPI_K3) { if (threadIdx.x >= 64) sfrag[threadIdx.x] = __ldg(a.frag2 + threadIdx.x - 64); }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane >> 2, t = lane & 3;
  int blk = blockIdx.y;
  const int stride = gridDim.x * NW;
  const float sg = (float)a.sg;
  HsConst hsk;
  { const uint32_t p = a.sg > 0 ? 0x3c003c00u : 0xbc00bc00u, q = a.sg > 0 ? 0xbc003c00u : 0x3c00bc00u;   // half2 (lo, hi) = (sg, sg), (sg, -sg)
    hsk.P = p; hsk.N = p ^ 0x80008000u; hsk.Q = q; hsk.R = q ^ 0x80008000u; }
  float part = 0.f;

  // per-block-row base pointers (64-bit once per Dirichlet block); everything below is 32-bit offsets in units of uint4
  const uint4 *in4, *aux4 = nullptr, *dot4 = nullptr;
  uint4 *out4, *out24 = nullptr;
  const uint32_t* lk32;
  const uint8_t* flp;
  const int* nbr = a.nbr;
  auto set_block = [&](int b) {
    blk = b;
    in4 = reinterpret_cast<const uint4*>(a.in) + (long)b * a.in_stride * (LS * 3);
    out4 = reinterpret_cast<uint4*>(a.out) + (long)b * a.out_stride * (LS * 3);
    if (EPI == EPI_K3) out24 = reinterpret_cast<uint4*>(a.out2) + (long)b * a.out2_stride * (LS * 3);
    if (EPI != EPI_PLAIN) aux4 = reinterpret_cast<const uint4*>(a.aux) + (long)b * a.aux_stride * (LS * 3);
    if (EPI == EPI_XPAY && a.dot_out) dot4 = reinterpret_cast<const uint4*>(a.dotv) + (long)b * a.dotv_stride * (LS * 3);
    lk32 = reinterpret_cast<const uint32_t*>(a.links) + (long)b * a.link_stride * (4 * NG);
    flp = a.flip + (long)b * a.link_stride;
  };

  // lane constants: fragment offset inside a site column (pad lanes clamped onto valid data, they meet zeros in B)
  const int tt = t < 3 ? t : 2;
  const int g0 = g < Cfg::N0 ? g : Cfg::N0 - 1;
  const int g1 = Cfg::NSEG == 2 ? (g < Cfg::N1 ? g : Cfg::N1 - 1) : 0;
  const int fo0 = g0 * 3 + tt, fo1 = 24 + g1 * 3 + tt;             // uint4 units
  const bool st0 = t < 3 && g < Cfg::N0, st1 = Cfg::NSEG == 2 && t < 3 && g < Cfg::N1;
  const int lko = ((g >> 1) * 3 + tt);                              // link word of this lane
  const bool lk_mine = t < 3 && g < 6 && (NG == 18 || (g >> 1) < 2);
  const uint32_t bsel = (g & 1) ? 0x1032u : 0x7610u;

  unsigned char* wsm = smraw + warp * SM::WARP;
  const uint32_t stage_u32 = smem_u32(wsm);
  const uint32_t bar_u32 = stage_u32 + 2 * SM::STAGE;
  {  // zero the stages once (absent neighbours are never copied), init the two mbarriers
    uint4* z = reinterpret_cast<uint4*>(wsm);
    for (int i = lane; i < 2 * SM::STAGE / 16; i += 32) z[i] = make_uint4(0, 0, 0, 0);
    if (lane == 0) { mbar_init(bar_u32, 1); mbar_init(bar_u32 + 8, 1); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    __syncwarp();
  }

  struct Meta { int nbv; uint32_t lk[8]; unsigned fl; };
  auto ld_meta = [&](int st, Meta& m) {
    const bool ok = st < a.n_out;
    m.nbv = (ok && lane < 8) ? __ldg(nbr + st * 8 + lane) : -1;
    m.fl = ok ? (unsigned)__ldg(flp + st) : 0u;
    const uint32_t* lk = lk32 + st * (4 * NG) + lko;
#pragma unroll
    for (int d = 0; d < 8; d++) m.lk[d] = (ok && lk_mine) ? __ldg(lk + d * (NG / 2)) : 0u;
  };
  // the xpay operand of the site itself: loaded at the top of a step, consumed in its epilogue (the hop hides the latency)
  auto ld_aux = [&](int st, uint4 (&x)[NSEG]) {
    if (EPI != EPI_PLAIN) {
      const bool ok = st < a.n_aux;
      const uint4* p = aux4 + st * (LS * 3);
      x[0] = (ok && st0) ? __ldg(p + fo0) : make_uint4(0, 0, 0, 0);
      if (NSEG == 2) x[NSEG - 1] = (ok && st1) ? __ldg(p + fo1) : make_uint4(0, 0, 0, 0);
    }
  };
  // issue the eight neighbour copies of the site whose table is m.nbv into stage `stg`
  auto issue = [&](const Meta& m, int stg) {
    const bool v = lane < 8 && m.nbv >= 0 && m.nbv < a.n_in_limit;
    const unsigned mask = __ballot_sync(0xffffffffu, v);
    const uint32_t bar = bar_u32 + 8 * stg;
    if (lane == 0) mbar_expect_tx(bar, (uint32_t)__popc(mask) * SM::SLOT);
    __syncwarp();
    if (v) bulk_g2s(stage_u32 + stg * SM::STAGE + lane * SM::SLOT, in4 + (long)m.nbv * (LS * 3), SM::SLOT, bar);
  };

  auto step = [&](int site, int stg, uint32_t parity, Meta& cur, const Meta& nxt) {
    const int far = site + 2 * stride;
    uint4 dv[NSEG], av[NSEG];
    ld_aux(site, av);
    if (EPI == EPI_XPAY && dot4 != nullptr) {
      const uint4* p = dot4 + site * (LS * 3);
      dv[0] = st0 ? __ldg(p + fo0) : make_uint4(0, 0, 0, 0);
      if (NSEG == 2) dv[NSEG - 1] = st1 ? __ldg(p + fo1) : make_uint4(0, 0, 0, 0);
    }
    issue(nxt, stg ^ 1);                       // site + stride (a harmless empty transaction past the end)
    const unsigned have = __ballot_sync(0xffffffffu, cur.nbv >= 0 && cur.nbv < a.n_in_limit) & 0xffu;
    uint32_t bfr[8];
#pragma unroll
    for (int d = 0; d < 8; d++) {
      uint32_t w = link_bfrag<NG>(cur.lk[d], g, t, bsel);
      if (d >= 6) { if ((cur.fl >> d) & 1u) w ^= 0x80008000u; }   // only time links cross the antiperiodic boundary (R7)
      bfr[d] = (have & (1u << d)) ? w : 0u;                       // absent neighbour: its slot holds stale data
    }
    ld_meta(far, cur);

    float S[NMT][4];
#pragma unroll
    for (int m = 0; m < NMT; m++) { S[m][0] = S[m][1] = S[m][2] = S[m][3] = 0.f; }
    mbar_wait(bar_u32 + 8 * stg, parity);
    // 128-bit shared-memory reads: the chunk {u0, l0, u1, l1} of colour t at s = g (and 8 + g), conflict free
    const uint32_t sb = stage_u32 + stg * SM::STAGE;
#define MSPCG_HOP_MU(MU)                                                                       \
    if (have & (3u << (2 * MU))) {                                                             \
      uint4 Ff[NSEG], Bb[NSEG];                                                                \
      const uint32_t pf = sb + (2 * MU) * SM::SLOT, pb = pf + SM::SLOT;                        \
      Ff[0] = lds128v(pf + 16 * fo0); Bb[0] = lds128v(pb + 16 * fo0);                          \
      if (NSEG == 2) { Ff[NSEG - 1] = lds128v(pf + 16 * fo1); Bb[NSEG - 1] = lds128v(pb + 16 * fo1); } \
      hop_mu_hs<MU, LS>(S, Ff, Bb, bfr[2 * MU], bfr[2 * MU + 1], sg, hsk);                     \
    }
    MSPCG_HOP_MU(0) MSPCG_HOP_MU(1) MSPCG_HOP_MU(2) MSPCG_HOP_MU(3)
#undef MSPCG_HOP_MU
    __syncwarp();                              // the stage may be overwritten by the copies issued in the next step

    dense5d_mma<LS>(S, sfrag, lane);

    uint4 o[NSEG];
    uint4* po = out4 + site * (LS * 3);
    if (EPI == EPI_PLAIN) {
      float_to_frag<LS>(S, o);
      if (st0) po[fo0] = o[0];
      if (NSEG == 2) { if (st1) po[fo1] = o[NSEG - 1]; }
    } else {
      float V[NMT][4];
      frag_to_float<LS>(av, V);
#pragma unroll
      for (int m = 0; m < NMT; m++) {
#pragma unroll
        for (int q = 0; q < 4; q++) S[m][q] = V[m][q] - S[m][q];
      }
      float_to_frag<LS>(S, o);
      if (EPI == EPI_K3) {
        if (site < a.n_out2) {
          uint4* p2 = out24 + site * (LS * 3);
          if (st0) p2[fo0] = o[0];
          if (NSEG == 2) { if (st1) p2[fo1] = o[NSEG - 1]; }
        }
        dense5d_mma<LS>(S, sfrag + 64, lane);
        float_to_frag<LS>(S, o);
      }
      if (st0) po[fo0] = o[0];
      if (NSEG == 2) { if (st1) po[fo1] = o[NSEG - 1]; }
      if (EPI == EPI_XPAY && dot4 != nullptr) {
        float P[NMT][4];
        frag_to_float<LS>(dv, P);
        if (st0 || st1) {
#pragma unroll
          for (int m = 0; m < NMT; m++) {
#pragma unroll
            for (int q = 0; q < 4; q++) part += P[m][q] * S[m][q];
          }
        }
      }
    }
  };

  // Thread blocks are persistent over Dirichlet blocks too (grid.y <= nblk): with thousands of small blocks (8^4 blocks of the
  // 48^3 x 96 lattice) one wave of resident thread blocks walks all of them.  ph0 / ph1: parity of the next phase to wait for
  // on the two stage barriers; an issue for a site past the end is an empty phase that nobody waits for and is skipped here.
  const int site0 = blockIdx.x * NW + warp;
  uint32_t ph0 = 0, ph1 = 0;
  for (int b = blockIdx.y; b < a.nblk; b += gridDim.y) {
    set_block(b);
    part = 0.f;
    Meta mA, mB;
    ld_meta(site0, mA); ld_meta(site0 + stride, mB);
    issue(mA, 0);
    int nst = 0;
    for (int site = site0; site < a.n_out; site += 2 * stride) {
      step(site, 0, ph0, mA, mB); ph0 ^= 1u; nst++;
      if (site + stride < a.n_out) { step(site + stride, 1, ph1, mB, mA); ph1 ^= 1u; nst++; }
    }
    if (nst == 0 || (nst & 1) == 0) ph0 ^= 1u; else ph1 ^= 1u;   // the trailing empty phase
    __syncwarp();

    if (EPI == EPI_XPAY) {
      if (a.dot_out != nullptr) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        __syncthreads();                       // red[] of the previous Dirichlet block has been read
        if (lane == 0) red[warp] = (double)part;
        __syncthreads();
        if (threadIdx.x == 0) {
          double tot = 0;
#pragma unroll
          for (int w = 0; w < NW; w++) tot += red[w];
          atomicAdd(a.dot_out + (long)blk * a.dot_stride, tot);
        }
      }
    }
  }
}

}  // namespace mspcg
