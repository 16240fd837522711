// hop_tile.cuh -- the fused hop kernel for fp16 storage as a thread-block-cooperative TILE kernel (the preconditioner's
// hot path; "the vector is loaded once into shared memory and reused by the stencil").
//
// k_hop_mma (hop_mma.cuh) gives every warp a private copy of the eight neighbour columns of its site: every input column
// crosses L2 -> SM eight times, and at Ls = 16 (768 B per column) the kernel runs at the L2 slice throughput
// (~12 TB/s) and not at the HBM roofline.  Here a persistent thread block owns a TILE of <= 32 output sites that are compact
// in 4D (tile_tables.hpp) and stages the UNION of their neighbour columns once (<= 128 columns, 4.0 per output site on a
// 4x4x2x2 cell instead of 8):
//   * warps 0..NWP-1 are producers: for every tile they issue one TMA bulk copy (cp.async.bulk, SASS UBLKCP) per RUN of
//     consecutive input columns (the lists are cell-ordered, geometry.hpp, so a 4x4x2x2 cell needs ~20 copies for its 128
//     columns), one per run of output sites for their links, and one for the tile header, all completing on the stage's
//     `full` mbarrier; two stages, so the copies of tile i+1 run while tile i is computed (a single warp issues a copy
//     every ~45 cycles -- lane-serialised ELECT / R2UR / UBLKCP -- hence several producer warps);
//   * the other NWC warps are consumers: warp w computes output sites w, w+NWC, ... of the tile with the arithmetic of
//     hop_mma.cuh (half-spinor projection, SU(3) x half-spinor and the Ls x Ls matrices on the tensor cores with
//     mma.m16n8k16, fp32 accumulation); neighbour fragments are 128-bit shared-memory reads at slot * column size;
//     link words are 32-bit shared-memory reads; a consumer touches global memory only for the xpay / dot operands
//     and for its stores.  When a warp is done with a stage it arrives on the stage's `empty` mbarrier.
// Tiles are dealt to thread blocks round robin over the flattened (Dirichlet block, tile) index (neighbouring cells are in
// flight at the same time: L2 reuse); the fused <p, A p> costs one atomic per warp and tile.
// Links carry the antiperiodic sign already (18 reals; the 12-real format keeps the per-warp kernel).
#pragma once
#include <type_traits>
#include "tile_tables.hpp"

namespace mspcg {

#ifndef MSPCG_TILE_NSTAGE
#define MSPCG_TILE_NSTAGE 2   // a third stage fits only for Ls <= 8 (59 KB per stage); measured there: -6 % in kernels 2/4, 0 in 3 and 5
#endif
#ifndef MSPCG_TILE_NWC_PLAIN
#define MSPCG_TILE_NWC_PLAIN 16
#endif
#ifndef MSPCG_TILE_NWP_PLAIN
#define MSPCG_TILE_NWP_PLAIN 4
#endif
template <int LS, int EPI = 0> struct TileCfg {
  enum {
    TS = TILE_TS, NIN = TILE_NIN, NSTAGE = MSPCG_TILE_NSTAGE,
    NWC = MSPCG_TILE_NWC_PLAIN,                     // consumer warps
    PAIR = (MSPCG_TILE_NWC_PLAIN <= 12),            // two sites per warp in one instruction stream (needs 128 registers: at most 12 + 4 warps)
    NWP = MSPCG_TILE_NWP_PLAIN,                     // producer warps
    COL = LS * 48,                       // bytes of one site column
    LINKREC = 8 * 18 * 2,                // bytes of the eight links of one output site
    OFF_ZERO = NIN * COL,                // one column of zeros: the slot of every absent neighbour (and of the pad lanes' link words)
    OFF_LINK = OFF_ZERO + COL,
    OFF_HDR = OFF_LINK + TS * LINKREC,
    STAGE = ((OFF_HDR + TILE_HDR + 127) / 128) * 128,
    SMEM = NSTAGE * STAGE,
    THREADS = 32 * (NWC + NWP),
  };
};

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint2 lds64(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];\n" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}

// (1 + c gamma_mu) psi = (h, h') with the half spinors h = u + c G l and h' = l + c G^dag u = c G^dag h  (G = -i sigma_k, 1 for mu = t;
// c = -sg forward, +sg backward; chunk = {u0, l0, u1, l1}).  h is formed in the lane (project_hs, hop_mma.cuh) and is the A fragment of
// upper += W h.  The lower half spinor is taken from the upper one: h' = c G^dag h, and G^dag = i sigma_k is a permutation of the two spin rows
// times a phase, so  lower += W h' = (c phase W) (rows of h permuted, one row negated for mu = y, z):  the phase and the sign c go into a
// second B fragment of the link (vf, vb: one byte permute each per direction and SITE), the row permutation is a choice of registers.
//   mu = x: h' = c i (h1, h0)    mu = y: h' = c (h1, -h0)    mu = z: h' = c i (h0, -h1)    mu = t: h' = c (h0, h1)
// Against projecting both half spinors in the lane this saves 32 packed fp16 FMAs and 16 permutes per site column, against mapping
// W_b h_b - W_f h_f onto the lower components after the MMA (hop_mma.cuh) 64 FMAs; h' is exact given h.
template <int MU, int LS>
__device__ __forceinline__ void hop_mu_perm(float (&S)[MmaCfg<LS>::NMT][4], const uint4 (&F)[MmaCfg<LS>::NSEG], const uint4 (&B)[MmaCfg<LS>::NSEG],
                                            uint32_t bf, uint32_t bb, uint32_t vf, uint32_t vb, const HsConst& k) {
#pragma unroll
  for (int seg = 0; seg < MmaCfg<LS>::NSEG; seg++) {
    uint32_t f0, f1, b0, b1;
    project_hs<MU, true>(F[seg], k, f0, f1);
    project_hs<MU, false>(B[seg], k, b0, b1);
    float (&S0)[4] = S[2 * seg], (&S1)[4] = S[2 * seg + 1];
    mma16816_4(S0[0], S0[1], S1[0], S1[1], f0, f1, b0, b1, bf, bb);
    if (MU == 0)      mma16816_4(S0[2], S0[3], S1[2], S1[3], f1, f0, b1, b0, vf, vb);
    else if (MU == 1) mma16816_4(S0[2], S0[3], S1[2], S1[3], f1, f0 ^ 0x80008000u, b1, b0 ^ 0x80008000u, vf, vb);
    else if (MU == 2) mma16816_4(S0[2], S0[3], S1[2], S1[3], f0, f1 ^ 0x80008000u, b0, b1 ^ 0x80008000u, vf, vb);
    else              mma16816_4(S0[2], S0[3], S1[2], S1[3], f0, f1, b0, b1, vf, vb);
  }
}

// dense5d_mma (hop_mma.cuh) with the A fragments of the two chirality blocks in registers instead of shared memory
template <int LS>
__device__ __forceinline__ void dense5d_mma_reg(float (&X)[MmaCfg<LS>::NMT][4], const uint4& A0, const uint4& A1) {
  typedef MmaCfg<LS> Cfg;
#pragma unroll
  for (int hi = 0; hi < 2; hi++) {
    const uint4& A = hi ? A1 : A0;
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

template <int LS, int EPI>
__global__ void __launch_bounds__(TileCfg<LS, EPI>::THREADS, 1) k_hop_tile(const HopArgs<__half> a) {
  typedef MmaCfg<LS> Cfg;
  typedef TileCfg<LS, EPI> TC;
  constexpr int NSEG = Cfg::NSEG, NMT = Cfg::NMT, NWC = TC::NWC;
  extern __shared__ __align__(128) unsigned char smraw[];
  __shared__ uint4 sfrag[EPI == EPI_K3 ? 128 : 64];       // A fragments of the 5D matrices (kernels 2 and 4 keep theirs in registers; the others have none to spare)
  __shared__ __align__(8) uint64_t bars[2 * TC::NSTAGE];  // full[stage], empty[stage]
  if (EPI != EPI_PLAIN) {
    if (threadIdx.x < 64) sfrag[threadIdx.x] = __ldg(a.frag1 + threadIdx.x);
    else if (EPI == EPI_K3 && threadIdx.x < 128) sfrag[threadIdx.x] = __ldg(a.frag2 + threadIdx.x - 64);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t sm_u32 = smem_u32(smraw);
  const uint32_t full_u32 = smem_u32(bars), empty_u32 = full_u32 + 8 * TC::NSTAGE;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < TC::NSTAGE; s++) { mbar_init(full_u32 + 8 * s, TC::NWP); mbar_init(empty_u32 + 8 * s, NWC); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();

  // Thread block b takes the tiles b, b + gridDim.x, ... of the flattened (Dirichlet block, tile) index: at any time the resident thread
  // blocks work on ~gridDim.x CONSECUTIVE tiles, i.e. on neighbouring cells, so a column shared by two tiles is fetched by both within
  // a few microseconds and the second fetch hits L2 (measured at C2 against contiguous chunks per thread block: DRAM reads -13 .. -22 %,
  // kernel time -3 .. -5 %, profiles/r2_hop_tile_whatif.md).
  const long total = (long)a.nblk * a.n_tiles;
  const long t_begin = blockIdx.x, t_step = gridDim.x;

  if (warp < TC::NWP) {
    // ----------------------------------------------------------------------------------------------- producer warps
    // Warp w fetches the input slots [w NIN/NWP, (w+1) NIN/NWP) (a lane issues a copy for each of its slots where a run starts)
    // and the link records of the output sites [w TS/NWP, (w+1) TS/NWP); warp 0 also fetches the tile header.  Every producer warp posts
    // the bytes of its own copies on the stage's `full` barrier (arrival count NWP) before it issues them.
    int stage = 0;
    uint32_t phases = 0xffffffffu;   // bit s: parity to wait for on empty[s]; a fresh barrier passes a wait on the phase before its first one
    constexpr int SPW = TC::NIN / TC::NWP / 32;        // input slots per lane
    constexpr int OPW = TC::TS / TC::NWP;              // output sites per producer warp
    const int slot0 = (TC::NIN / TC::NWP) * warp + lane, oj = OPW * warp + (lane < OPW ? lane : 0);
    for (long tt = t_begin; tt < total; tt += t_step) {
      const int blk = (int)(tt / a.n_tiles), ti = (int)(tt - (long)blk * a.n_tiles);
      const TileRec* rec = a.tiles + ti;
      int col[SPW]; uint32_t run[SPW], nrun = 0;
#pragma unroll
      for (int q = 0; q < SPW; q++) { col[q] = __ldg(rec->in_col + slot0 + 32 * q); run[q] = __ldg(rec->in_run + slot0 + 32 * q); nrun += run[q]; }
      const int osite = __ldg(rec->out_site + oj);
      const uint32_t orun = lane < OPW ? (uint32_t)__ldg(rec->out_run + oj) : 0u;
      const uint32_t sb = sm_u32 + stage * TC::STAGE, bar = full_u32 + 8 * stage;
      const uint32_t bytes = __reduce_add_sync(0xffffffffu, nrun) * TC::COL + __reduce_add_sync(0xffffffffu, orun) * TC::LINKREC + (warp == 0 ? TILE_HDR : 0);
      mbar_wait(empty_u32 + 8 * stage, (phases >> stage) & 1u);
      if (lane == 0) {
        mbar_expect_tx(bar, bytes);
        if (warp == 0) bulk_g2s(sb + TC::OFF_HDR, rec, TILE_HDR, bar);
      }
      __syncwarp();
      const unsigned char* inb = reinterpret_cast<const unsigned char*>(a.in) + (long)blk * a.in_stride * TC::COL;
#pragma unroll
      for (int q = 0; q < SPW; q++)
        if (run[q]) bulk_g2s(sb + (slot0 + 32 * q) * TC::COL, inb + (long)col[q] * TC::COL, run[q] * TC::COL, bar);
      if (orun)
        bulk_g2s(sb + TC::OFF_LINK + oj * TC::LINKREC,
                 reinterpret_cast<const unsigned char*>(a.links) + ((long)blk * a.link_stride + osite) * TC::LINKREC, orun * TC::LINKREC, bar);
      // kernel 3's consumers read the xpay operand of the output sites straight from global memory about one tile later: pull it into L2 now
      // (measured at C2: kernel 3 -4 %; the same for kernel 5's two operands changes nothing, and prefetching the NEXT tile's columns makes
      // every kernel slower, +3 .. +15 %: profiles/r2_hop_tile_whatif.md)
      if (EPI == EPI_K3 && orun) {
        const int n = osite + (int)orun <= a.n_aux ? (int)orun : a.n_aux - osite;
        if (n > 0) bulk_prefetch_l2(reinterpret_cast<const unsigned char*>(a.aux) + ((long)blk * a.aux_stride + osite) * TC::COL, n * TC::COL);
      }
      phases ^= 1u << stage;
      stage = stage + 1 == TC::NSTAGE ? 0 : stage + 1;
    }
    return;
  }

  // -------------------------------------------------------------------------------------------------- consumer warps
  const int cw = warp - TC::NWP;
  const int g = lane >> 2, t = lane & 3;
  HsConst hsk;
  { const uint32_t p = a.sg > 0 ? 0x3c003c00u : 0xbc00bc00u, q = a.sg > 0 ? 0xbc003c00u : 0x3c00bc00u;   // half2 (sg, sg), (sg, -sg)
    hsk.P = p; hsk.N = p ^ 0x80008000u; hsk.Q = q; hsk.R = q ^ 0x80008000u; }
  // lane constants: fragment offset inside a site column (pad lanes clamped onto valid data, they meet zeros in B)
  const int tt3 = t < 3 ? t : 2;
  const int g0 = g < Cfg::N0 ? g : Cfg::N0 - 1;
  const int g1 = Cfg::NSEG == 2 ? (g < Cfg::N1 ? g : Cfg::N1 - 1) : 0;
  const int fo0 = g0 * 3 + tt3, fo1 = 24 + g1 * 3 + tt3;             // uint4 units
  const bool st0 = t < 3 && g < Cfg::N0, st1 = Cfg::NSEG == 2 && t < 3 && g < Cfg::N1;
  const bool lk_mine = t < 3 && g < 6;
  const uint32_t lk_off = (uint32_t)(lk_mine ? ((g >> 1) * 3 + t) : 0);   // this lane's word inside an 18-real link
  // B fragments by one byte permute of (raw, N), raw = (Wr, Wi) the lane's complex link entry, N = -raw.  Lanes with even g hold the real
  // output column (Xr, -Xi) of a matrix X, odd g the imaginary one (Xi, Xr):
  //   X = W: (Wr, -Wi) | (Wi, Wr)     X = -W: (-Wr, Wi) | (-Wi, -Wr)     X = iW: (-Wi, -Wr) | (Wr, -Wi)     X = -iW: (Wi, Wr) | (-Wr, Wi)
  const bool odd = (g & 1) != 0;
  const uint32_t bsel = odd ? 0x1032u : 0x7610u;
  const uint32_t sel_p = bsel, sel_m = odd ? 0x5476u : 0x3254u, sel_ip = odd ? 0x7610u : 0x5476u, sel_im = odd ? 0x3254u : 0x1032u;
  const bool sgp = a.sg > 0;                   // c = -sg forward, +sg backward
  const uint32_t vsel_f13 = sgp ? sel_m : sel_p, vsel_b13 = sgp ? sel_p : sel_m;      // mu = y, t: c W
  const uint32_t vsel_f02 = sgp ? sel_im : sel_ip, vsel_b02 = sgp ? sel_ip : sel_im;  // mu = x, z: c i W
  const int lk_step = lk_mine ? 9 : 0;

  uint4 rA0 = make_uint4(0, 0, 0, 0), rA1 = rA0;
  if (EPI == EPI_PLAIN) { rA0 = __ldg(a.frag1 + lane); rA1 = __ldg(a.frag1 + 32 + lane); }
  float part = 0.f;
  int part_blk = -1;
  auto flush_dot = [&]() {
    if (EPI == EPI_XPAY && a.dot_out != nullptr && part_blk >= 0) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
      if (lane == 0) atomicAdd(a.dot_out + (long)part_blk * a.dot_stride, (double)part);
    }
    part = 0.f;
  };

  int stage = 0;
  uint32_t phases = 0u;              // bit s: parity to wait for on full[s]
  {  // the zero column of both stages (never touched by the copies)
    for (int s2 = 0; s2 < TC::NSTAGE; s2++) {
      uint4* z = reinterpret_cast<uint4*>(smraw + s2 * TC::STAGE + TC::OFF_ZERO);
      for (int i = threadIdx.x - 32 * TC::NWP; i < TC::COL / 16; i += 32 * NWC) z[i] = make_uint4(0, 0, 0, 0);
    }
    asm volatile("bar.sync 1, %0;\n" ::"n"(32 * NWC) : "memory");   // consumer warps only
  }
  int rot = 0;
  for (long tt = t_begin; tt < total; tt += t_step) {
    const int blk = (int)(tt / a.n_tiles);
    if (blk != part_blk) { flush_dot(); part_blk = blk; }
    const uint4* aux4 = nullptr; const uint4* dot4 = nullptr;
    uint4* out4 = reinterpret_cast<uint4*>(a.out) + (long)blk * a.out_stride * (LS * 3);
    uint4* out24 = nullptr;
    if (EPI == EPI_K3) out24 = reinterpret_cast<uint4*>(a.out2) + (long)blk * a.out2_stride * (LS * 3);
    if (EPI != EPI_PLAIN) aux4 = reinterpret_cast<const uint4*>(a.aux) + (long)blk * a.aux_stride * (LS * 3);
    if (EPI == EPI_XPAY && a.dot_out) dot4 = reinterpret_cast<const uint4*>(a.dotv) + (long)blk * a.dotv_stride * (LS * 3);

    const uint32_t sb = sm_u32 + stage * TC::STAGE;
    mbar_wait(full_u32 + 8 * stage, (phases >> stage) & 1u);
    const uint32_t hdr = sb + TC::OFF_HDR;
    const uint4* stg4 = reinterpret_cast<const uint4*>(smraw + stage * TC::STAGE);
    const uint32_t* lk32 = reinterpret_cast<const uint32_t*>(smraw + stage * TC::STAGE + TC::OFF_LINK);
    const uint32_t* zero32 = reinterpret_cast<const uint32_t*>(smraw + stage * TC::STAGE + TC::OFF_ZERO);
    const int n_out = (int)lds32(hdr);
    // One output site in three pieces, so that two sites can be worked on in the same straight-line code (TC::PAIR, below).  Measured at C2
    // (DESIGN.md section 4): 12 consumer warps x 2 sites per warp run exactly as fast as 16 x 1 (K2/K4 0.0727 vs 0.0723 ms), as do 20 and 24
    // warps at 80 / 72 registers -- the kernel is bound by its per-site instruction stream on the ALU / FMA pipes, not by latency.
    struct SiteCtx { int site; uint2 sl; unsigned have; uint4 av[NSEG], dv[NSEG]; float S[NMT][4]; const uint32_t* lkb; };
    auto begin = [&](SiteCtx& x, const int j) {
      x.site = (int)lds32(hdr + 16 + 4 * j);
      x.sl = lds64(hdr + 16 + 4 * TC::TS + 8 * j);
      x.have = (lds32(hdr + 16 + 12 * TC::TS + (j & ~3)) >> (8 * (j & 3))) & 0xffu;
      if (EPI != EPI_PLAIN) {
        const bool ok = x.site < a.n_aux;
        const uint4* p = aux4 + (long)x.site * (LS * 3);
        x.av[0] = (ok && st0) ? __ldg(p + fo0) : make_uint4(0, 0, 0, 0);
        if (NSEG == 2) x.av[NSEG - 1] = (ok && st1) ? __ldg(p + fo1) : make_uint4(0, 0, 0, 0);
      }
      if (EPI == EPI_XPAY && dot4 != nullptr) {
        const uint4* p = dot4 + (long)x.site * (LS * 3);
        x.dv[0] = st0 ? __ldg(p + fo0) : make_uint4(0, 0, 0, 0);
        if (NSEG == 2) x.dv[NSEG - 1] = st1 ? __ldg(p + fo1) : make_uint4(0, 0, 0, 0);
      }
      x.lkb = lk_mine ? lk32 + j * (TC::LINKREC / 4) + lk_off : zero32;   // pad lanes read zeros
#pragma unroll
      for (int m = 0; m < NMT; m++) { x.S[m][0] = x.S[m][1] = x.S[m][2] = x.S[m][3] = 0.f; }
    };
    // direction pair MU: B fragments of the two links (this lane's complex entry as (Wr, -Wi) or (Wi, Wr), and the phase-carrying
    // variant for the lower components), the two neighbour columns from their slots, projections and MMAs
    auto hop_mu = [&](auto mu_tag, SiteCtx& x) {
      constexpr int MU = decltype(mu_tag)::value;
      uint32_t bf[2], bv[2];
#pragma unroll
      for (int bw = 0; bw < 2; bw++) {
        const uint32_t raw = x.lkb[(2 * MU + bw) * lk_step], neg = raw ^ 0x80008000u;
        bf[bw] = __byte_perm(raw, neg, bsel);
        bv[bw] = __byte_perm(raw, neg, (MU & 1) ? (bw ? vsel_b13 : vsel_f13) : (bw ? vsel_b02 : vsel_f02));
      }
      uint4 Ff[NSEG], Bb[NSEG];
      const uint32_t w2 = (MU < 2 ? x.sl.x : x.sl.y) >> (16 * (MU & 1));
      const uint4* pf = stg4 + (w2 & 0xffu) * (TC::COL / 16);
      const uint4* pb = stg4 + ((w2 >> 8) & 0xffu) * (TC::COL / 16);
      Ff[0] = pf[fo0]; Bb[0] = pb[fo0];
      if (NSEG == 2) { Ff[NSEG - 1] = pf[fo1]; Bb[NSEG - 1] = pb[fo1]; }
      hop_mu_perm<MU, LS>(x.S, Ff, Bb, bf[0], bf[1], bv[0], bv[1], hsk);
    };
    auto finish = [&](SiteCtx& x) {
      float (&S)[NMT][4] = x.S;
      const int site = x.site;
      if (EPI == EPI_PLAIN) dense5d_mma_reg<LS>(S, rA0, rA1);
      else dense5d_mma<LS>(S, sfrag, lane);
      uint4 o[NSEG];
      uint4* po = out4 + (long)site * (LS * 3);
      if (EPI == EPI_PLAIN) {
        float_to_frag<LS>(S, o);
        if (st0) po[fo0] = o[0];
        if (NSEG == 2) { if (st1) po[fo1] = o[NSEG - 1]; }
      } else {
        float V[NMT][4];
        frag_to_float<LS>(x.av, V);
#pragma unroll
        for (int m = 0; m < NMT; m++) {
#pragma unroll
          for (int q = 0; q < 4; q++) S[m][q] = V[m][q] - S[m][q];
        }
        float_to_frag<LS>(S, o);
        if (EPI == EPI_K3) {
          if (site < a.n_out2) {
            uint4* p2 = out24 + (long)site * (LS * 3);
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
          frag_to_float<LS>(x.dv, P);
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
    typedef std::integral_constant<int, 0> M0; typedef std::integral_constant<int, 1> M1;
    typedef std::integral_constant<int, 2> M2; typedef std::integral_constant<int, 3> M3;
    // sites are dealt to the consumer warps round robin, continuing across tiles (tile sizes are not multiples of NWC)
    int j = cw >= rot ? cw - rot : cw - rot + NWC;
    if (lds32(hdr + 8) != 0u) {
      // every site of the tile has all eight neighbours (flag in the tile header): no branches, two sites at a time
      for (; TC::PAIR && j + NWC < n_out; j += 2 * NWC) {
        SiteCtx x0, x1;
        begin(x0, j); begin(x1, j + NWC);
        hop_mu(M0(), x0); hop_mu(M0(), x1); hop_mu(M1(), x0); hop_mu(M1(), x1);
        hop_mu(M2(), x0); hop_mu(M2(), x1); hop_mu(M3(), x0); hop_mu(M3(), x1);
        finish(x0); finish(x1);
      }
      for (; j < n_out; j += NWC) {
        SiteCtx x0;
        begin(x0, j);
        hop_mu(M0(), x0); hop_mu(M1(), x0); hop_mu(M2(), x0); hop_mu(M3(), x0);
        finish(x0);
      }
    } else {
      // halo tiles of a Dirichlet block: direction pairs with no neighbour are skipped (a single absent neighbour reads the zero column)
      for (; j < n_out; j += NWC) {
        SiteCtx x0;
        begin(x0, j);
        if (x0.have & 0x03u) hop_mu(M0(), x0);
        if (x0.have & 0x0cu) hop_mu(M1(), x0);
        if (x0.have & 0x30u) hop_mu(M2(), x0);
        if (x0.have & 0xc0u) hop_mu(M3(), x0);
        finish(x0);
      }
    }
    rot = (rot + n_out) % NWC;
    __syncwarp();
    if (lane == 0) mbar_arrive(empty_u32 + 8 * stage);
    phases ^= 1u << stage;
    stage = stage + 1 == TC::NSTAGE ? 0 : stage + 1;
  }
  flush_dot();
}

}  // namespace mspcg
