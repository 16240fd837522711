// dense5d_tma.cuh -- the dense fifth-dimension contraction (M5^-1, M5^-dag or any pair of Ls x Ls chirality blocks; PAPER.md:260-264,
// 272; north_star item 2) on an fp16 NATIVE vector as a warp-specialised, persistent tcgen05 GEMM fed and drained
// by tensor-map TMA.
//
//   out[site][s][colour][j] = sum_s' M_hi(j)[s][s'] in[site][s'][colour][j],   j = (sp, hi, re/im) = the 8 halves of a 16-byte chunk.
//
// Per colour this is D[site][n] = sum_k A[site][k] B[n][k] with k = (s', j'), n = (s, j), B[n][k] = M_hi(j)[s][s'] delta_jj'.
// The tcgen05 A operand wants 8-row x 16-byte core matrices (K-major, no swizzle); in HBM the 16-byte chunk of (site, s', colour)
// is 48 Ls bytes away from the next site's.  A 4D tensor map with the dimension ORDER (chunk, site, s', colour) -- strides 48 Ls,
// 48 and 16 bytes -- makes the TMA unit do the permutation: the box (8, 128, Ls, 3) lands in shared memory as [colour][s'][site][16 B],
// i.e. for every colour a valid canonical operand with SBO = 128 B (next 8 sites) and LBO = 2 KB (next s'), and the same map on
// the output vector stores the result tile.  One UTMALDG and one UTMASTG of 96 KB (Ls = 16) per 128-site tile.
//
// Roles (192 threads): warp 0 lane 0 issues the tile loads (2 stages); warp 1 lane 0 issues 3 x Ls/2 tcgen05.mma (128 x 8Ls x 16,
// fp32 accumulators in tensor memory, 4 accumulator slots in rotation) and commits them to mbarriers; warps 2-5 are the epilogue:
// thread = TMEM lane = site row, tcgen05.ld of its 8 Ls accumulator columns, round to fp16, write the chunk back INTO the stage the
// operand came from (the MMAs of that colour are complete), and after the third colour one thread issues the TMA store and frees
// the stage when the store has read it.  Ragged last tile: TMA zero-fills loads and clips stores.
#pragma once
#include <cuda.h>

namespace mspcg {

struct Dense5dTmaArgs {
  const float* M;     // [hi][s][s'] the two chirality blocks (fp32; rounded to fp16 in the kernel)
  long n_sites;
};

template <int LS> struct Dense5dTmaCfg {
  enum {
    N = 8 * LS, K = 8 * LS, NSTAGE = 2, NACC = 4,
    A_COLOUR = 128 * LS * 16,            // bytes of one colour of a tile: [s'][site][16 B]
    STAGE = 3 * A_COLOUR,
    B_BYTES = N * K * 2,
    OFF_B = NSTAGE * STAGE,
    OFF_BAR = OFF_B + B_BYTES,
    SMEM = OFF_BAR + 128,
    TMEM_COLS = (NACC * N <= 256 ? 256 : 512),
    THREADS = 192,
  };
};

namespace tma {
__device__ __forceinline__ void load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];\n"
               ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}
__device__ __forceinline__ void store_4d(const CUtensorMap* map, int c0, int c1, int c2, int c3, uint32_t src) {
  asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4}], [%5];\n"
               ::"l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(src) : "memory");
}
__device__ __forceinline__ void store_commit_and_wait_read() {
  asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
  asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory");
}
__device__ __forceinline__ void store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;\n" ::: "memory"); }
__device__ __forceinline__ void ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]),
        "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]),
        "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
}
}  // namespace tma

template <int LS>
__global__ void __launch_bounds__(Dense5dTmaCfg<LS>::THREADS, 1)
k_dense5d_tma(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_out, const Dense5dTmaArgs a) {
  typedef Dense5dTmaCfg<LS> DC;
  extern __shared__ __align__(128) unsigned char dsm[];
  __shared__ uint32_t tmem_slot;
  const uint32_t sm0 = (uint32_t)__cvta_generic_to_shared(dsm);
  const uint32_t bars = sm0 + DC::OFF_BAR;
  // barriers: full[2] | stage_free[2] | acc_full[4] | acc_free[4]
  const uint32_t full = bars, sfree = bars + 16, accfull = bars + 32, accfree = bars + 64;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const long n_tiles = (a.n_sites + 127) / 128;
  const long my_tiles = blockIdx.x < n_tiles ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

  if (warp == 1) tc::tmem_alloc<DC::TMEM_COLS>(&tmem_slot);
  if (tid == 0) {
    for (int i = 0; i < DC::NSTAGE; i++) { mbar_init(full + 8 * i, 1); mbar_init(sfree + 8 * i, 1); }
    for (int i = 0; i < DC::NACC; i++) { mbar_init(accfull + 8 * i, 1); mbar_init(accfree + 8 * i, 4); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  // B operand built in place from the two Ls x Ls chirality blocks: core matrix (s, s') = diag_j M_hi(j)[s][s']
  {
    unsigned char* Bs = dsm + DC::OFF_B;
    for (int pr = tid; pr < LS * LS; pr += DC::THREADS) {
      const uint32_t m0 = (uint32_t)__half_as_ushort(__float2half_rn(__ldg(a.M + pr)));
      const uint32_t m1 = (uint32_t)__half_as_ushort(__float2half_rn(__ldg(a.M + LS * LS + pr)));
      uint4* d = reinterpret_cast<uint4*>(Bs) + pr * 8;
      d[0] = make_uint4(m0, 0, 0, 0); d[1] = make_uint4(m0 << 16, 0, 0, 0); d[2] = make_uint4(0, m1, 0, 0); d[3] = make_uint4(0, m1 << 16, 0, 0);
      d[4] = make_uint4(0, 0, m0, 0); d[5] = make_uint4(0, 0, m0 << 16, 0); d[6] = make_uint4(0, 0, 0, m1); d[7] = make_uint4(0, 0, 0, m1 << 16);
    }
  }
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;

  if (warp == 0) {
    // ------------------------------------------------------------------------------------------------- TMA load producer
    if (lane == 0) {
      for (long i = 0; i < my_tiles; i++) {
        const int st = (int)(i % DC::NSTAGE);
        const uint32_t use = (uint32_t)(i / DC::NSTAGE);
        mbar_wait(sfree + 8 * st, (use & 1u) ^ 1u);          // passes at once on the first use of a stage
        const long site0 = ((long)blockIdx.x + i * gridDim.x) * 128;
        mbar_expect_tx(full + 8 * st, (uint32_t)DC::STAGE);
        tma::load_4d(sm0 + st * DC::STAGE, &tm_in, 0, (int)site0, 0, 0, full + 8 * st);
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------------------------------------------ MMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = tc::idesc_f16(128, DC::N);
      const uint32_t b0 = sm0 + DC::OFF_B;
      long q = 0;
      for (long i = 0; i < my_tiles; i++) {
        const int st = (int)(i % DC::NSTAGE);
        mbar_wait(full + 8 * st, (uint32_t)((i / DC::NSTAGE) & 1));
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
        for (int c = 0; c < 3; c++, q++) {
          const int slot = (int)(q % DC::NACC);
          mbar_wait(accfree + 8 * slot, (uint32_t)(((q / DC::NACC) & 1) ^ 1));   // epilogue has drained this accumulator
          asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
          const uint32_t a0 = sm0 + st * DC::STAGE + c * DC::A_COLOUR;
#pragma unroll
          for (int kk = 0; kk < DC::K / 16; kk++)
            tc::mma_f16(tmem + slot * DC::N, tc::smem_desc(a0 + kk * 2 * 2048, 2048, 128), tc::smem_desc(b0 + kk * 256, 128, LS * 128), idesc, kk > 0);
          tc::commit(accfull + 8 * slot);
        }
      }
    }
  } else {
    // -------------------------------------------------------------------------------------------------- epilogue warps
    const int quad = warp & 3;                         // TMEM lanes 32*quad .. 32*quad+31
    const int row = quad * 32 + lane;                  // site row of the tile
    long q = 0;
    for (long i = 0; i < my_tiles; i++) {
      const int st = (int)(i % DC::NSTAGE);
      unsigned char* stage = dsm + st * DC::STAGE;
      for (int c = 0; c < 3; c++, q++) {
        const int slot = (int)(q % DC::NACC);
        mbar_wait(accfull + 8 * slot, (uint32_t)((q / DC::NACC) & 1));
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
        uint4* dst = reinterpret_cast<uint4*>(stage + c * DC::A_COLOUR) + row;     // + s * 128 chunks
#pragma unroll
        for (int s4 = 0; s4 < LS; s4 += 4) {
          uint32_t v[32];
          tma::ld32(tmem + ((uint32_t)(quad * 32) << 16) + slot * DC::N + s4 * 8, v);
#pragma unroll
          for (int u = 0; u < 4; u++) {
            uint4 o;
            o.x = pack_h2(__uint_as_float(v[8 * u]), __uint_as_float(v[8 * u + 1])); o.y = pack_h2(__uint_as_float(v[8 * u + 2]), __uint_as_float(v[8 * u + 3]));
            o.z = pack_h2(__uint_as_float(v[8 * u + 4]), __uint_as_float(v[8 * u + 5])); o.w = pack_h2(__uint_as_float(v[8 * u + 6]), __uint_as_float(v[8 * u + 7]));
            dst[(s4 + u) * 128] = o;
          }
        }
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(accfree + 8 * slot);
      }
      // all three colours of the tile are back in the stage: publish the generic-proxy writes to the async proxy, store, free the stage
      asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
      asm volatile("bar.sync 1, 128;\n" ::: "memory");
      if (tid == 64) {
        const long site0 = ((long)blockIdx.x + i * gridDim.x) * 128;
        tma::store_4d(&tm_out, 0, (int)site0, 0, 0, sm0 + st * DC::STAGE);
        tma::store_commit_and_wait_read();
        mbar_arrive(sfree + 8 * st);
      }
    }
    if (tid == 64) tma::store_wait_all();
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 1) tc::tmem_free<DC::TMEM_COLS>(tmem);
}

}  // namespace mspcg
