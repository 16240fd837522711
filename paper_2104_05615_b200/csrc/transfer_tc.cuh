// transfer_tc.cuh -- the reduced-Ls transfer matrices T and T^dag (eq. 20-21) as
// dense contractions on the 5th-generation tensor cores: tcgen05.mma (kind::f16, fp16 operands, fp32 accumulation in
// tensor memory), issued by one thread, operands in shared memory in the canonical K-major no-swizzle layout.
//
// T is the identity in colour and 4D site, so for every colour the contraction is a GEMM
//     D[site][n] = sum_k A[site][k] B[n][k]
// forward  (rhat = T r / scale):    k = (s, spin, re/im) 8*Ls,   n = (a, sp, hi, re/im) 8*Lh
// backward (z = scale T^dag x + mu r):  k = (a, spin, re/im) 8*Lh,  n = (s, spin, re/im) 8*Ls
// with B the real 2x2-block form of the complex matrix (host-built, fp16).  A thread block owns a tile of 128 sites:
// M = 128 rows = sites, one accumulator of N columns per colour (3 N <= 384 of the 512 TMEM columns).
//
// Shared-memory operand layout (UMMA canonical, K-major, SWIZZLE_NONE): element (row r, k) at
//     (r / 8) * SBO + (k / 8) * LBO + (r % 8) * 16 + (k % 8) * 2   bytes,
// i.e. 8-row x 16-byte core matrices.  The 8 reals (spin, re/im) of one (site, s, colour) are exactly one 16-byte
// core-matrix row, so a thread that holds the 24 reals of (site, s) writes three 128-bit shared-memory stores.
// A uses LBO = 144 (16 bytes of padding between K-adjacent core matrices: conflict-free stores from lanes that
// differ in s), B uses LBO = 128 (a linear copy of the host image).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace mspcg {

namespace tc {

__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
  uint64_t d = 0;
  d |= (uint64_t)((addr & 0x3FFFFu) >> 4);          // start address, bits [0,14)
  d |= (uint64_t)((lbo >> 4) & 0x3FFFu) << 16;      // leading-dimension byte offset (K-adjacent core matrices)
  d |= (uint64_t)((sbo >> 4) & 0x3FFFu) << 32;      // stride byte offset (8-row groups)
  d |= (uint64_t)1 << 46;                           // descriptor version (sm_100)
  return d;                                         // base offset 0, layout type 0 = SWIZZLE_NONE
}
// kind::f16 instruction descriptor: D fp32, A and B fp16, both K-major, M x N.
__host__ __device__ constexpr uint32_t idesc_f16(int M, int N) {
  return (1u << 4) | (0u << 7) | (0u << 10) | (0u << 15) | (0u << 16) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void mma_f16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void ld8(uint32_t taddr, float (&v)[8]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
  for (int i = 0; i < 8; i++) v[i] = __uint_as_float(r[i]);
}
template <int NCOLS> __device__ __forceinline__ void tmem_alloc(uint32_t* slot_smem) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"((uint32_t)__cvta_generic_to_shared(slot_smem)), "n"(NCOLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
}
template <int NCOLS> __device__ __forceinline__ void tmem_free(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(taddr), "n"(NCOLS) : "memory");
}

constexpr int TILE = 128;        // sites per thread block = MMA M
constexpr int A_LBO = 144;       // bytes between K-adjacent core matrices of A (128 + 16 padding)

}  // namespace tc

struct TransferArgs {
  const void* in;       // forward: r_in (TIO, Ls)      backward: xhat (TX = float, Lh)
  const void* rin;      // backward: r_in (TIO, Ls) for the mu term
  void* out;            // forward: rhat (__half, Lh)   backward: z (TIO, Ls)
  const __half* Bimg;   // device image of the B operand [N/8][K/8][8 rows][8 halfs]
  long n_sites;         // sites per block (nE0)
  const float* scale;   // per-block max-abs scale (R14)
  double* rho0;         // forward: rho0[blk] += |rhat|^2
  double mu;
};

// KG = number of 8-wide K groups (forward: Ls, backward: Lh); NG8 = N / 8 (forward: Lh, backward: Ls).
template <int KG, int NG8> struct TransferCfg {
  enum { K = 8 * KG, N = 8 * NG8, A_SBO = KG * tc::A_LBO, A_COLOUR = 16 * A_SBO, B_BYTES = N * K * 2,
         TMEM_COLS = (3 * N <= 32 ? 32 : (3 * N <= 64 ? 64 : (3 * N <= 128 ? 128 : (3 * N <= 256 ? 256 : 512)))),
         SMEM = 3 * A_COLOUR + B_BYTES + 64 };
};

// Forward transfer, fp16 inner storage: rhat = T (r_in / scale), rho0 += |rhat|^2.   grid = (ceil(n_sites/128), nblk).
template <typename TIO, int LS, int LH>
__global__ void __launch_bounds__(128, 1) k_reduce_begin_tc(const TransferArgs a) {
  typedef TransferCfg<LS, LH> Cfg;
  extern __shared__ __align__(128) unsigned char tsm[];
  __shared__ uint32_t tmem_slot;
  __shared__ double red[32];
  unsigned char* As = tsm;
  unsigned char* Bs = tsm + 3 * Cfg::A_COLOUR;
  const uint32_t bar = (uint32_t)__cvta_generic_to_shared(tsm + 3 * Cfg::A_COLOUR + Cfg::B_BYTES);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int blk = blockIdx.y;
  const long site0 = (long)blockIdx.x * tc::TILE;
  const TIO* rin = reinterpret_cast<const TIO*>(a.in);
  const float f = 1.f / (float)blk_scale(a.scale, blk);

  if (warp == 0) tc::tmem_alloc<Cfg::TMEM_COLS>(&tmem_slot);
  if (tid == 0) { mbar_init(bar, 1); asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
  // B image: linear copy
  for (int i = tid; i < Cfg::B_BYTES / 16; i += 128) reinterpret_cast<uint4*>(Bs)[i] = __ldg(reinterpret_cast<const uint4*>(a.Bimg) + i);
  // A tiles: thread handles (site, s) pairs, s fastest
  for (int idx = tid; idx < tc::TILE * LS; idx += 128) {
    const int r = idx / LS, s = idx - r * LS;
    const long site = site0 + r;
    float v[24];
    if (site < a.n_sites) {
      typename ST<TIO>::C w[24];
      load24<TIO>(rin, (long)blk * a.n_sites + site, s, LS, w);
#pragma unroll
      for (int k = 0; k < 24; k++) v[k] = (float)w[k] * f;
    } else {
#pragma unroll
      for (int k = 0; k < 24; k++) v[k] = 0.f;
    }
    unsigned char* dst = As + (r >> 3) * Cfg::A_SBO + s * tc::A_LBO + (r & 7) * 16;
#pragma unroll
    for (int c = 0; c < 3; c++) {   // chunk of colour c: (spin 0..3) x (re, im)
      uint4 q;
      q.x = pack_h2(v[(0 * 3 + c) * 2], v[(0 * 3 + c) * 2 + 1]); q.y = pack_h2(v[(1 * 3 + c) * 2], v[(1 * 3 + c) * 2 + 1]);
      q.z = pack_h2(v[(2 * 3 + c) * 2], v[(2 * 3 + c) * 2 + 1]); q.w = pack_h2(v[(3 * 3 + c) * 2], v[(3 * 3 + c) * 2 + 1]);
      *reinterpret_cast<uint4*>(dst + c * Cfg::A_COLOUR) = q;
    }
  }
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // generic-proxy smem writes -> visible to the MMA (async proxy)
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;
  if (tid == 0) {
    const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(As), b0 = (uint32_t)__cvta_generic_to_shared(Bs);
    constexpr uint32_t idesc = tc::idesc_f16(128, Cfg::N);
#pragma unroll
    for (int c = 0; c < 3; c++)
#pragma unroll
      for (int kk = 0; kk < Cfg::K / 16; kk++)
        tc::mma_f16(tmem + c * Cfg::N, tc::smem_desc(a0 + c * Cfg::A_COLOUR + kk * 2 * tc::A_LBO, tc::A_LBO, Cfg::A_SBO),
                    tc::smem_desc(b0 + kk * 256, 128, LS * 128), idesc, kk > 0);
    tc::commit(bar);
  }
  mbar_wait(bar, 0);
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  // epilogue: thread = TMEM lane = site row; per colour and s_hat one 16-byte chunk (sp, hi, re/im) of the fp16 layout
  const int r = tid;
  const long site = site0 + r;
  double part = 0;
  uint4* out4 = reinterpret_cast<uint4*>(a.out) + ((long)blk * a.n_sites + site) * (LH * 3);
#pragma unroll
  for (int c = 0; c < 3; c++)
#pragma unroll
    for (int ah = 0; ah < LH; ah++) {
      float v[8];
      tc::ld8(tmem + ((uint32_t)(warp * 32) << 16) + c * Cfg::N + ah * 8, v);
      uint4 q;
      q.x = pack_h2(v[0], v[1]); q.y = pack_h2(v[2], v[3]); q.z = pack_h2(v[4], v[5]); q.w = pack_h2(v[6], v[7]);
      if (site < a.n_sites) {
        out4[ah * 3 + c] = q;
        const uint32_t u[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int i = 0; i < 4; i++) { const float2 h = unpack_h2(u[i]); part += (double)h.x * h.x + (double)h.y * h.y; }
      }
    }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  const double tot = block_sum(part, red, tid, 128);   // contains a __syncthreads
  if (tid == 0 && tot != 0.0) atomicAdd(a.rho0 + blk, tot);
  if (warp == 0) tc::tmem_free<Cfg::TMEM_COLS>(tmem);
  (void)lane;
}

// Backward transfer: z = scale * T^dag xhat + mu * r_in, xhat fp32 (Lh), z and r_in in TIO (Ls).
template <typename TIO, int LS, int LH>
__global__ void __launch_bounds__(128, 1) k_reduce_end_tc(const TransferArgs a) {
  typedef TransferCfg<LH, LS> Cfg;   // K = 8*Lh, N = 8*Ls
  extern __shared__ __align__(128) unsigned char tsm[];
  __shared__ uint32_t tmem_slot;
  unsigned char* As = tsm;
  unsigned char* Bs = tsm + 3 * Cfg::A_COLOUR;
  const uint32_t bar = (uint32_t)__cvta_generic_to_shared(tsm + 3 * Cfg::A_COLOUR + Cfg::B_BYTES);
  const int tid = threadIdx.x, warp = tid >> 5;
  const int blk = blockIdx.y;
  const long site0 = (long)blockIdx.x * tc::TILE;
  const float* xh = reinterpret_cast<const float*>(a.in);
  const TIO* rin = reinterpret_cast<const TIO*>(a.rin);
  TIO* z = reinterpret_cast<TIO*>(a.out);

  if (warp == 0) tc::tmem_alloc<Cfg::TMEM_COLS>(&tmem_slot);
  if (tid == 0) { mbar_init(bar, 1); asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
  for (int i = tid; i < Cfg::B_BYTES / 16; i += 128) reinterpret_cast<uint4*>(Bs)[i] = __ldg(reinterpret_cast<const uint4*>(a.Bimg) + i);
  for (int idx = tid; idx < tc::TILE * LH; idx += 128) {
    const int r = idx / LH, s = idx - r * LH;
    const long site = site0 + r;
    float v[24];
    if (site < a.n_sites) load24<float>(xh, (long)blk * a.n_sites + site, s, LH, v);
    else {
#pragma unroll
      for (int k = 0; k < 24; k++) v[k] = 0.f;
    }
    unsigned char* dst = As + (r >> 3) * Cfg::A_SBO + s * tc::A_LBO + (r & 7) * 16;
#pragma unroll
    for (int c = 0; c < 3; c++) {
      uint4 q;
      q.x = pack_h2(v[(0 * 3 + c) * 2], v[(0 * 3 + c) * 2 + 1]); q.y = pack_h2(v[(1 * 3 + c) * 2], v[(1 * 3 + c) * 2 + 1]);
      q.z = pack_h2(v[(2 * 3 + c) * 2], v[(2 * 3 + c) * 2 + 1]); q.w = pack_h2(v[(3 * 3 + c) * 2], v[(3 * 3 + c) * 2 + 1]);
      *reinterpret_cast<uint4*>(dst + c * Cfg::A_COLOUR) = q;
    }
  }
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;
  if (tid == 0) {
    const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(As), b0 = (uint32_t)__cvta_generic_to_shared(Bs);
    constexpr uint32_t idesc = tc::idesc_f16(128, Cfg::N);
#pragma unroll
    for (int c = 0; c < 3; c++)
#pragma unroll
      for (int kk = 0; kk < Cfg::K / 16; kk++)
        tc::mma_f16(tmem + c * Cfg::N, tc::smem_desc(a0 + c * Cfg::A_COLOUR + kk * 2 * tc::A_LBO, tc::A_LBO, Cfg::A_SBO),
                    tc::smem_desc(b0 + kk * 256, 128, LH * 128), idesc, kk > 0);
    tc::commit(bar);
  }
  mbar_wait(bar, 0);
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const long site = site0 + tid;
  const double f = blk_scale(a.scale, blk);
  for (int s = 0; s < LS; s++) {
    float d[3][8];
#pragma unroll
    for (int c = 0; c < 3; c++) tc::ld8(tmem + ((uint32_t)(warp * 32) << 16) + c * Cfg::N + s * 8, d[c]);
    if (site < a.n_sites) {
      const long gs = (long)blk * a.n_sites + site;
      typename ST<TIO>::C rr[24], o[24];
      load24<TIO>(rin, gs, s, LS, rr);
#pragma unroll
      for (int sp = 0; sp < 4; sp++)
#pragma unroll
        for (int c = 0; c < 3; c++)
#pragma unroll
          for (int ri = 0; ri < 2; ri++) {
            const int k = (sp * 3 + c) * 2 + ri;
            o[k] = (typename ST<TIO>::C)(f * (double)d[c][sp * 2 + ri] + a.mu * (double)rr[k]);
          }
      store24<TIO>(z, gs, s, LS, o);
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tc::tmem_free<Cfg::TMEM_COLS>(tmem);
}

// ---------------------------------------------------------------------------------------------------------------
// The dense fifth-dimension contraction M5^-1 / M5^-dag as a stand-alone tcgen05 GEMM (
// north_star item 2): out[s][n] = sum_s' M_hi[s][s'] in[s'][n] on an fp16 NATIVE vector (layout of hop_mma.cuh:
// v[site][s][colour][sp][hi][re,im]).  Per colour it is the GEMM  D[site][n] = sum_k A[site][k] B[n][k]  with
// k = (s', j), n = (s, j), j = (sp, hi, re/im) the eight halves of one 16-byte chunk, and B[n][k] = M_hi[s][s'] delta_jj'
// (real, built in shared memory by the kernel).  The 16-byte chunk of one (site, s', colour) in HBM IS one core-matrix row of the K-major
// canonical layout, so the A tile is filled with plain 128-bit copies, no conversion.  M = 128 sites per thread block,
// N = K = 8 Ls, an N-column fp32 accumulator in tensor memory; the MMA does 8x the minimal flop count
// (the delta_jj' zeros), which the tensor pipe does not notice at this size.
// Inside the fused hop kernels the same contraction runs on register fragments (mma.sync, hop_mma.cuh); this kernel
// serves the places where M5^-1 stands alone on an fp16 vector.
struct Dense5dTcArgs {
  const uint4* in; uint4* out;   // NATIVE fp16 vectors, n_sites site columns of Ls*3 chunks
  const float* M;                // [hi][s][s'] the two chirality blocks of the matrix (fp32; rounded to fp16 in the kernel)
  long n_sites;
};
template <int LS> struct Dense5dTcCfg {
  enum { N = 8 * LS, TMEM_COLS = (2 * N <= 32 ? 32 : (2 * N <= 64 ? 64 : (2 * N <= 128 ? 128 : (2 * N <= 256 ? 256 : 512)))),
         SMEM = 2 * TransferCfg<LS, LS>::A_COLOUR + TransferCfg<LS, LS>::B_BYTES + 64 };
};
// Persistent thread blocks (grid = min(tiles, 2 per SM)); a work item is (tile of 128 sites, colour).  Two A tiles and two
// accumulators: the 16-byte chunks of item q+1 are fetched with cp.async (no registers, no wait) while the MMAs, the tensor-memory
// read-back and the stores of item q run.  B is built once per thread block.
template <int LS>
__global__ void __launch_bounds__(128, 2) k_dense5d_tc(const Dense5dTcArgs a) {
  typedef TransferCfg<LS, LS> Cfg;
  typedef Dense5dTcCfg<LS> DC;
  extern __shared__ __align__(128) unsigned char tsm[];
  __shared__ uint32_t tmem_slot;
  unsigned char* Bs = tsm + 2 * Cfg::A_COLOUR;
  const uint32_t as_u32 = (uint32_t)__cvta_generic_to_shared(tsm);
  const uint32_t bar = (uint32_t)__cvta_generic_to_shared(tsm + 2 * Cfg::A_COLOUR + Cfg::B_BYTES);
  const int tid = threadIdx.x, warp = tid >> 5;
  const long n_tiles = (a.n_sites + tc::TILE - 1) / tc::TILE;
  const long my_tiles = blockIdx.x < n_tiles ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const long Q = 3 * my_tiles;

  if (warp == 0) tc::tmem_alloc<DC::TMEM_COLS>(&tmem_slot);
  if (tid == 0) { mbar_init(bar, 1); mbar_init(bar + 8, 1); asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
  // B operand built in place from the two Ls x Ls chirality blocks (every thread block reading a 32 KB image from the same L2 lines
  // was a hot spot): core matrix (s, s') = diag_j M_hi(j)[s][s'], row j is one 16-byte store with a single non-zero half.
  for (int pr = tid; pr < LS * LS; pr += 128) {
    const uint32_t m0 = (uint32_t)__half_as_ushort(__float2half_rn(__ldg(a.M + pr)));
    const uint32_t m1 = (uint32_t)__half_as_ushort(__float2half_rn(__ldg(a.M + LS * LS + pr)));
    uint4* d = reinterpret_cast<uint4*>(Bs) + pr * 8;
    d[0] = make_uint4(m0, 0, 0, 0); d[1] = make_uint4(m0 << 16, 0, 0, 0); d[2] = make_uint4(0, m1, 0, 0); d[3] = make_uint4(0, m1 << 16, 0, 0);
    d[4] = make_uint4(0, 0, m0, 0); d[5] = make_uint4(0, 0, m0 << 16, 0); d[6] = make_uint4(0, 0, 0, m1); d[7] = make_uint4(0, 0, 0, m1 << 16);
  }
  // asynchronous fetch of item q into A tile q & 1 (one commit group per item, empty past the end)
  auto fetch = [&](long q) {
    if (q < Q) {
      const long site0 = ((long)blockIdx.x + (q / 3) * gridDim.x) * tc::TILE;
      const int c = (int)(q % 3);
      const uint32_t buf = as_u32 + (uint32_t)(q & 1) * Cfg::A_COLOUR;
#pragma unroll
      for (int i = 0; i < LS; i++) {
        const int idx = tid + i * 128, r = idx / LS, s = idx - r * LS;
        const long st = site0 + r;
        const uint32_t dst = buf + (r >> 3) * Cfg::A_SBO + s * tc::A_LBO + (r & 7) * 16;
        if (st < a.n_sites) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(a.in + st * (LS * 3) + s * 3 + c) : "memory");
        else asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};\n" ::"r"(dst), "r"(0u) : "memory");
      }
    }
    asm volatile("cp.async.commit_group;\n" ::: "memory");
  };
  fetch(0);
  for (long q = 0; q < Q; q++) {
    fetch(q + 1);                                    // its A tile was read by the MMAs of item q - 1, waited for below
    asm volatile("cp.async.wait_group 1;\n" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const uint32_t tmem = tmem_slot + (uint32_t)(q & 1) * Cfg::N;
    const uint32_t bq = bar + 8 * (uint32_t)(q & 1);
    if (tid == 0) {
      const uint32_t a0 = as_u32 + (uint32_t)(q & 1) * Cfg::A_COLOUR, b0 = (uint32_t)__cvta_generic_to_shared(Bs);
      constexpr uint32_t idesc = tc::idesc_f16(128, Cfg::N);
#pragma unroll
      for (int kk = 0; kk < Cfg::K / 16; kk++)
        tc::mma_f16(tmem, tc::smem_desc(a0 + kk * 2 * tc::A_LBO, tc::A_LBO, Cfg::A_SBO), tc::smem_desc(b0 + kk * 256, 128, LS * 128), idesc, kk > 0);
      tc::commit(bq);
    }
    mbar_wait(bq, (uint32_t)((q >> 1) & 1));
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const long site = ((long)blockIdx.x + (q / 3) * gridDim.x) * tc::TILE + tid;   // thread = TMEM lane = site row
    const int c = (int)(q % 3);
    uint4* out4 = a.out + site * (LS * 3);
#pragma unroll
    for (int s = 0; s < LS; s++) {
      float v[8];
      tc::ld8(tmem + ((uint32_t)(warp * 32) << 16) + s * 8, v);
      uint4 o;
      o.x = pack_h2(v[0], v[1]); o.y = pack_h2(v[2], v[3]); o.z = pack_h2(v[4], v[5]); o.w = pack_h2(v[6], v[7]);
      if (site < a.n_sites) out4[s * 3 + c] = o;
    }
  }
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tc::tmem_free<DC::TMEM_COLS>(tmem_slot);
}

}  // namespace mspcg
