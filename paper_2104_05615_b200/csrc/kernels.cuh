// kernels.cuh -- sm_100a device code of libmspcg.
//
// Data layout in HBM ("site slab"): a vector on a site list is
//     v[site][chunk][s][16 bytes]
// i.e. for every 4D site the whole fifth-dimension column is one contiguous slab of Ls*24 reals; a 16-byte chunk
// holds 2 (fp64) / 4 (fp32) / 8 (fp16) consecutive reals of the 24 (index (spin*3+colour)*2+reim) of one (site, s).
// A thread block owns NS consecutive sites x all Ls; thread (j, s).  Lanes that differ in s read consecutive
// 16-byte chunks (Ls*16 contiguous bytes per site), so every neighbour fetch is a fully used, 128-bit vectorised,
// coalesced access whatever the 4D geometry of the neighbour; the links of the NS sites are one contiguous record
// staged once per block in shared memory.  The hop result never leaves the SM before the fifth-dimension matrices
// are applied to it (shared-memory slab), which is the fusion of PAPER.md:249-258 (eq. 16).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

#include "site_math.cuh"
#include "tile_tables.hpp"

namespace mspcg {

// ------------------------------------------------------------------------------------------------ storage traits
template <typename T> struct ST;
template <> struct ST<double> { typedef double C; typedef double2 V; typedef double2 P; enum { PER = 2, NCH = 12 }; };
template <> struct ST<float>  { typedef float C;  typedef float4 V;  typedef float2 P;  enum { PER = 4, NCH = 6 }; };
template <> struct ST<__half> { typedef float C;  typedef uint4 V;   typedef __half2 P; enum { PER = 8, NCH = 3 }; };

template <int LS> struct Tile { enum { NS = (LS >= 12 ? 8 : (LS >= 6 ? 16 : 32)), NT = NS * LS }; };

__device__ __forceinline__ void unpackV(const double2& q, double* v) { v[0] = q.x; v[1] = q.y; }
__device__ __forceinline__ void unpackV(const float4& q, float* v) { v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w; }
__device__ __forceinline__ void unpackV(const uint4& q, float* v) {
  const __half2* h = reinterpret_cast<const __half2*>(&q);
#pragma unroll
  for (int i = 0; i < 4; i++) { float2 f = __half22float2(h[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
}
__device__ __forceinline__ void packV(double2& q, const double* v) { q.x = v[0]; q.y = v[1]; }
__device__ __forceinline__ void packV(float4& q, const float* v) { q.x = v[0]; q.y = v[1]; q.z = v[2]; q.w = v[3]; }
__device__ __forceinline__ void packV(uint4& q, const float* v) {
  __half2* h = reinterpret_cast<__half2*>(&q);
#pragma unroll
  for (int i = 0; i < 4; i++) h[i] = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
}

// 24 reals of (site, s); `site` is the global site index in the array (block offset already added).
// fp64 / fp32: site-slab layout v[site][chunk][s][16 B].  fp16: v[site][s][colour][sp][hi][re,im] with spin = 2*hi+sp
// (48 contiguous bytes per (site, s); the fragment layout of hop_mma.cuh), chunk c = colour.
template <typename T> struct Lay {   // V-index of chunk c of (site, s) and position of real k inside the 24
  static __device__ __forceinline__ long idx(long site, int s, int LS, int c) { return (site * ST<T>::NCH + c) * LS + s; }
  static __device__ __forceinline__ int k(int c, int e) { return c * ST<T>::PER + e; }
};
template <> struct Lay<__half> {
  static __device__ __forceinline__ long idx(long site, int s, int LS, int c) { return (site * LS + s) * 3 + c; }
  // element e of the colour-c chunk: sp = e>>2, hi = (e>>1)&1, ri = e&1  ->  k = ((2*hi+sp)*3 + c)*2 + ri
  static __device__ __forceinline__ int k(int c, int e) { return ((2 * ((e >> 1) & 1) + (e >> 2)) * 3 + c) * 2 + (e & 1); }
};
template <typename T>
__device__ __forceinline__ void load24(const T* __restrict__ base, long site, int s, int LS, typename ST<T>::C* v) {
  typedef typename ST<T>::V V;
  const V* p = reinterpret_cast<const V*>(base);
#pragma unroll
  for (int c = 0; c < ST<T>::NCH; c++) {
    V q = __ldg(p + Lay<T>::idx(site, s, LS, c));
    typename ST<T>::C w[ST<T>::PER];
    unpackV(q, w);
#pragma unroll
    for (int e = 0; e < ST<T>::PER; e++) v[Lay<T>::k(c, e)] = w[e];
  }
}
template <typename T>
__device__ __forceinline__ void load24_pred(const T* __restrict__ base, long site, int s, int LS, bool ok, typename ST<T>::C* v) {
  if (ok) load24<T>(base, site, s, LS, v);
  else {
#pragma unroll
    for (int k = 0; k < 24; k++) v[k] = 0;
  }
}
template <typename T>
__device__ __forceinline__ void store24(T* __restrict__ base, long site, int s, int LS, const typename ST<T>::C* v) {
  typedef typename ST<T>::V V;
  V* p = reinterpret_cast<V*>(base);
#pragma unroll
  for (int c = 0; c < ST<T>::NCH; c++) {
    typename ST<T>::C w[ST<T>::PER];
#pragma unroll
    for (int e = 0; e < ST<T>::PER; e++) w[e] = v[Lay<T>::k(c, e)];
    V q; packV(q, w);
    p[Lay<T>::idx(site, s, LS, c)] = q;
  }
}

__device__ __forceinline__ double toD(double x) { return x; }
__device__ __forceinline__ double toD(float x) { return (double)x; }
__device__ __forceinline__ float ldreal(const float* p) { return __ldg(p); }
__device__ __forceinline__ double ldreal(const double* p) { return __ldg(p); }
__device__ __forceinline__ float ldreal(const __half* p) { return __half2float(__ldg(p)); }

// Block-wide sum of one double per thread; result valid in thread 0.  `red` holds >= 32 doubles of shared memory.
__device__ __forceinline__ double block_sum(double v, double* red, int tid, int nthreads) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = tid >> 5, nw = (nthreads + 31) >> 5;
  if ((tid & 31) == 0) red[w] = v;
  __syncthreads();
  double t = 0;
  if (tid == 0) for (int i = 0; i < nw; i++) t += red[i];
  return t;
}

// ------------------------------------------------------------------------ shared-memory geometry of one thread block
template <typename C, int LS> struct Smem {
  enum {
    NS = Tile<LS>::NS,
    UREC = (sizeof(C) == 4 ? 20 : 18),                 // reals per staged link (fp32: padded to 5 x 16 B)
    USTRIDE = 8 * UREC + (sizeof(C) == 4 ? 4 : 2),     // per-site stride, shifted by 16 B against bank aliasing
    SPAD = (((LS - 24 * LS) % 32) + 32) % 32,          // slab stride == LS (mod 32 banks): conflict-free
    SSTRIDE = 24 * LS + SPAD,
  };
};

// Fifth-dimension matrix on the slab: out[k] = sum_s' M[chir(k)][s][s'] * slab[k][s'],  chir = 0 for spin 0,1 (P+),
// 1 for spin 2,3 (P-).  Msm is stored transposed per chirality, Msm[ch][s'][s], so lanes read consecutive words.
// This is the dense Ls x Ls contraction of PAPER.md:260 on the ALUs.
template <typename C, int LS>
__device__ __forceinline__ void dense5d(const C* __restrict__ slab_j, const C* __restrict__ Msm, int s, C* out) {
  C m0[LS], m1[LS];
#pragma unroll
  for (int r = 0; r < LS; r++) { m0[r] = Msm[r * LS + s]; m1[r] = Msm[(LS + r) * LS + s]; }
#pragma unroll
  for (int k = 0; k < 24; k++) {
    const C* row = slab_j + k * LS;
    C a = 0;
    if (sizeof(C) == 4 && LS % 4 == 0) {
#pragma unroll
      for (int r = 0; r < LS; r += 4) {
        float4 q = *reinterpret_cast<const float4*>(row + r);
        if (k < 12) { a += m0[r] * (C)q.x; a += m0[r + 1] * (C)q.y; a += m0[r + 2] * (C)q.z; a += m0[r + 3] * (C)q.w; }
        else        { a += m1[r] * (C)q.x; a += m1[r + 1] * (C)q.y; a += m1[r + 2] * (C)q.z; a += m1[r + 3] * (C)q.w; }
      }
    } else {
#pragma unroll
      for (int r = 0; r < LS; r += 2) {
        C q0 = row[r], q1 = row[r + 1];
        if (k < 12) { a += m0[r] * q0; a += m0[r + 1] * q1; }
        else        { a += m1[r] * q0; a += m1[r + 1] * q1; }
      }
    }
    out[k] = a;
  }
}

// Stand-alone fifth-dimension matrix, out = M in on n_sites site columns (set-up steps of the full solve: the M5^-1
// factors of the prepared source, eq. 6, that are not preceded by a hop).  mat: [2][LS][LS] transposed per
// chirality like HopArgs::mat1.
template <typename T, int LS>
__global__ void __launch_bounds__(Tile<LS>::NT) k_dense5d(const T* __restrict__ in, T* __restrict__ out, const typename ST<T>::C* __restrict__ mat, long n_sites) {
  typedef typename ST<T>::C C;
  typedef Smem<C, LS> SM;
  constexpr int NS = Tile<LS>::NS;
  extern __shared__ __align__(16) unsigned char smraw[];
  C* slab = reinterpret_cast<C*>(smraw);
  C* Msm = slab + NS * SM::SSTRIDE;
  const int s = threadIdx.x, j = threadIdx.y;
  for (int i = j * LS + s; i < 2 * LS * LS; i += NS * LS) Msm[i] = mat[i];
  const long site = (long)blockIdx.x * NS + j;
  const bool live = site < n_sites;
  C v[24], o[24];
  load24_pred<T>(in, live ? site : 0, s, LS, live, v);
  C* slab_j = slab + j * SM::SSTRIDE;
#pragma unroll
  for (int k = 0; k < 24; k++) slab_j[k * LS + s] = v[k];
  __syncthreads();
  dense5d<C, LS>(slab_j, Msm, s, o);
  if (live) store24<T>(out, site, s, LS, o);
}

// ------------------------------------------------------------------------------------------ fused hop kernel (A3+A4)
template <typename T> struct HopArgs {
  typedef typename ST<T>::C C;
  const T* in;  long in_stride;  int n_in_limit;   // input list array [blk][in_stride sites]; neighbours >= limit are dropped
  T* out;       long out_stride;                   // [blk][out_stride]
  T* out2;      long out2_stride; int n_out2;      // K3: y written for sites < n_out2 into `out2`, w into `out`
  const T* aux; long aux_stride;  int n_aux;       // xpay operand (zero for sites >= n_aux)
  const T* dotv; long dotv_stride;                 // if dot_out: dot_out[blk*dot_stride] += Re<dotv, out>
  double* dot_out; int dot_stride;
  const int* nbr;                                  // [n_out][8], shared by all blocks
  const T* links; const uint8_t* flip; long link_stride;  // [blk][link_stride][8][ng], [blk][link_stride]
  int n_out, ng;
  int nblk;                                        // fp16 path: Dirichlet blocks to walk (grid.y may be smaller)
  const C* mat1; const C* mat2;                    // device [2][LS][LS], transposed per chirality
  const uint4* frag1; const uint4* frag2;          // fp16 path: the same matrices as mma A fragments [2][32] (hop_mma.cuh)
  const TileRec* tiles; int n_tiles;               // fp16 tile kernel (hop_tile.cuh): site tiles of this stage, shared by all blocks
  C sg;                                            // +1: D^w, -1: D^w^dag
};

enum { EPI_PLAIN = 0, EPI_K3 = 1, EPI_XPAY = 2 };

template <int MU, typename T, int LS>
__device__ __forceinline__ void hop_dir(typename ST<T>::C* acc, const T* __restrict__ in, long blk_off, int s,
                                        const int* nbs_j, const typename ST<T>::C* U_j, typename ST<T>::C sg) {
  typedef typename ST<T>::C C;
  typedef Smem<C, LS> SM;
#pragma unroll
  for (int bw = 0; bw < 2; bw++) {
    const int d = 2 * MU + bw;
    const int nb = nbs_j[d];
    C psi[24], W[18];
    load24_pred<T>(in, blk_off + (nb < 0 ? 0 : nb), s, LS, nb >= 0, psi);
    const C* u = U_j + d * SM::UREC;
    if (sizeof(C) == 4) {
#pragma unroll
      for (int q = 0; q < 4; q++) { float4 f = *reinterpret_cast<const float4*>(u + 4 * q); W[4 * q] = f.x; W[4 * q + 1] = f.y; W[4 * q + 2] = f.z; W[4 * q + 3] = f.w; }
      float2 f2 = *reinterpret_cast<const float2*>(u + 16); W[16] = f2.x; W[17] = f2.y;
    } else {
#pragma unroll
      for (int q = 0; q < 9; q++) { double2 f = *reinterpret_cast<const double2*>(u + 2 * q); W[2 * q] = f.x; W[2 * q + 1] = f.y; }
    }
    hop_term<MU, C>(acc, psi, W, bw ? sg : -sg);
  }
}

template <typename T, int LS, int EPI>
__global__ void __launch_bounds__(Tile<LS>::NT, (sizeof(typename ST<T>::C) == 8 ? 4 : 5)) k_hop(const HopArgs<T> a) {
  typedef typename ST<T>::C C;
  typedef Smem<C, LS> SM;
  constexpr int NS = Tile<LS>::NS, NT = Tile<LS>::NT;
  extern __shared__ __align__(16) unsigned char smraw[];
  C* Usm = reinterpret_cast<C*>(smraw);
  C* slab = Usm + NS * SM::USTRIDE;
  C* M1 = slab + NS * SM::SSTRIDE;
  C* M2 = M1 + 2 * LS * LS;
  int* nbs = reinterpret_cast<int*>(M2 + (EPI == EPI_K3 ? 2 * LS * LS : 0));
  __shared__ double red[32];

  const int s = threadIdx.x, j = threadIdx.y, tid = j * LS + s;
  const int blk = blockIdx.y;
  const int site0 = blockIdx.x * NS, site = site0 + j;
  const bool live = site < a.n_out;

  // ---- stage neighbour indices, links (convert, rebuild third row, fold the boundary sign) and matrices
  for (int l = tid; l < NS * 8; l += NT) {
    const int jj = l >> 3, d = l & 7, st = site0 + jj;
    C* u = Usm + jj * SM::USTRIDE + d * SM::UREC;
    int nb = -1;
    if (st < a.n_out) {
      nb = __ldg(a.nbr + (long)st * 8 + d);
      if (nb >= a.n_in_limit) nb = -1;
      const long ls = (long)blk * a.link_stride + st;
      const T* g = a.links + (ls * 8 + d) * a.ng;
      C W[18];
      for (int q = 0; q < a.ng; q++) W[q] = ldreal(g + q);
      if (a.ng == 12) su3_third_row(W);
      const C sgn = ((__ldg(a.flip + ls) >> d) & 1) ? (C)-1 : (C)1;
#pragma unroll
      for (int q = 0; q < 18; q++) u[q] = sgn * W[q];
    } else {
#pragma unroll
      for (int q = 0; q < 18; q++) u[q] = 0;
    }
    nbs[l] = nb;
  }
  for (int l = tid; l < 2 * LS * LS; l += NT) { M1[l] = a.mat1[l]; if (EPI == EPI_K3) M2[l] = a.mat2[l]; }
  __syncthreads();

  // ---- the Wilson hop for (site, s): eight neighbours (eq. 8)
  C acc[24];
#pragma unroll
  for (int k = 0; k < 24; k++) acc[k] = 0;
  {
    const long in_off = (long)blk * a.in_stride;
    const int* nbs_j = nbs + j * 8;
    const C* U_j = Usm + j * SM::USTRIDE;
    hop_dir<0, T, LS>(acc, a.in, in_off, s, nbs_j, U_j, a.sg);
    hop_dir<1, T, LS>(acc, a.in, in_off, s, nbs_j, U_j, a.sg);
    hop_dir<2, T, LS>(acc, a.in, in_off, s, nbs_j, U_j, a.sg);
    hop_dir<3, T, LS>(acc, a.in, in_off, s, nbs_j, U_j, a.sg);
  }

  // ---- fifth-dimension epilogue on the shared-memory slab
  C* slab_j = slab + j * SM::SSTRIDE;
#pragma unroll
  for (int k = 0; k < 24; k++) slab_j[k * LS + s] = acc[k];
  __syncthreads();
  C o[24];
  dense5d<C, LS>(slab_j, M1, s, o);

  if (EPI == EPI_PLAIN) {
    if (live) store24<T>(a.out, (long)blk * a.out_stride + site, s, LS, o);
    return;
  }
  // y = aux - M1 hop
  {
    C v[24];
    load24_pred<T>(a.aux, (long)blk * a.aux_stride + (site < a.n_aux ? site : 0), s, LS, live && site < a.n_aux, v);
#pragma unroll
    for (int k = 0; k < 24; k++) o[k] = v[k] - o[k];
  }
  if (EPI == EPI_K3) {
    if (live && site < a.n_out2) store24<T>(a.out2, (long)blk * a.out2_stride + site, s, LS, o);
    __syncthreads();  // everyone has finished reading the slab
#pragma unroll
    for (int k = 0; k < 24; k++) slab_j[k * LS + s] = o[k];
    __syncthreads();
    C w[24];
    dense5d<C, LS>(slab_j, M2, s, w);
    if (live) store24<T>(a.out, (long)blk * a.out_stride + site, s, LS, w);
    return;
  }
  // EPI_XPAY
  if (live) store24<T>(a.out, (long)blk * a.out_stride + site, s, LS, o);
  if (a.dot_out != nullptr) {
    double part = 0;
    if (live) {
      C p[24];
      load24<T>(a.dotv, (long)blk * a.dotv_stride + site, s, LS, p);
      C t = 0;
#pragma unroll
      for (int k = 0; k < 24; k++) t += p[k] * o[k];
      part = toD(t);
    }
    const double tot = block_sum(part, red, tid, NT);
    if (tid == 0) atomicAdd(a.dot_out + (long)blk * a.dot_stride, tot);
  }
}

}  // namespace mspcg
#include "hop_mma.cuh"
#include "hop_tile.cuh"
namespace mspcg {

// Fixed-point storage of PAPER.md:268-285 eq. 17 (reading R21) applied to the 24 reals of ONE colour-spinor, which is what a thread of the
// BLAS-1 kernels holds: v becomes what an 8- / 16-bit store of it returns,  integer / limit * scale  with scale = max |v| (fp32),
// integer = round-half-even(v / scale * limit), limit = 2^(bits-1) - 1; all in fp32, products and quotients rounded separately.
template <typename C> __device__ __forceinline__ void fixed_round24(C* v, int bits) {
  float m = 0.f;
#pragma unroll
  for (int k = 0; k < 24; k++) m = fmaxf(m, fabsf((float)v[k]));
  const float lim = bits == 8 ? 127.f : 32767.f;
  const float safe = m > 0.f ? m : 1.f;
#pragma unroll
  for (int k = 0; k < 24; k++) {
    const float q = rintf(__fmul_rn(__fdiv_rn((float)v[k], safe), lim));
    v[k] = m > 0.f ? (C)__fmul_rn(__fdiv_rn(q, lim), m) : (C)0;
  }
}

// ------------------------------------------------------------------ K1: Mphi (bidiagonal in s), fused with p-updates
// mode 0: t = Mphi in                                      (last item of eq. 16)
// mode 1: p = z + beta p (beta by value), t = Mphi p       (outer iteration, Algorithm 1 line "p = z + beta p")
// mode 2: inner CG of block blk, iteration `it`: p = r (it = 0) or r + (rho[it]/rho[it-1]) p, t = Mphi p  (R13)
template <typename T> struct MphiArgs {
  typedef typename ST<T>::C C;
  const T* in; T* p; T* t;          // mode 0: in -> t;  mode 1/2: in = z or r, p updated in place, t = Mphi p
  long n_sites;                     // sites per block (stride of all three arrays)
  int mode, it, nblk;
  double beta; const double* beta_dev;   // mode 1: beta by value, or read from device memory when beta_dev != null
  const double* rho; const double* pq;   // inner-CG scalars [it][nblk]
  C diag, off, mf;                  // Mphi = diag*1 + off*(P+ S_minus + P- S_plus), wrap factor -mf
  int fixed_bits;                   // fp32 storage only: p passes through the 8- / 16-bit fixed-point store of eq. 17 (0 = off)
};

// true while block `blk` has had rho > 0 and <p,q> > 0 in every iteration 0..it (reading R13: a block that hits
// rho == 0 or <p,Ap> <= 0 stops and keeps its current x).
__device__ __forceinline__ bool inner_alive(const double* rho, const double* pq, int nblk, int blk, int it) {
  bool ok = true;
  for (int i = 0; i <= it; i++) ok = ok && (rho[(long)i * nblk + blk] > 0.0) && (pq[(long)i * nblk + blk] > 0.0);
  return ok;
}

template <typename T, int LS>
__global__ void __launch_bounds__(Tile<LS>::NT) k_mphi(const MphiArgs<T> a) {
  typedef typename ST<T>::C C;
  typedef Smem<C, LS> SM;
  constexpr int NS = Tile<LS>::NS;
  extern __shared__ __align__(16) unsigned char smraw[];
  C* slab = reinterpret_cast<C*>(smraw);
  const int s = threadIdx.x, j = threadIdx.y;
  const int blk = blockIdx.y;
  const long site = (long)blockIdx.x * NS + j;
  const bool live = site < a.n_sites;
  const long gs = (long)blk * a.n_sites + (live ? site : 0);
  C v[24];
  load24_pred<T>(a.in, gs, s, LS, live, v);
  if (a.mode != 0) {
    C beta = 0;
    bool have_p = true;
    if (a.mode == 1) beta = a.beta_dev ? (C)*a.beta_dev : (C)a.beta;
    else if (a.it == 0) have_p = false;
    else {
      const bool ok = inner_alive(a.rho, a.pq, a.nblk, blk, a.it - 1);
      beta = ok ? (C)(a.rho[(long)a.it * a.nblk + blk] / a.rho[(long)(a.it - 1) * a.nblk + blk]) : (C)0;
    }
    if (have_p) {
      C p[24];
      load24_pred<T>(a.p, gs, s, LS, live, p);
#pragma unroll
      for (int k = 0; k < 24; k++) v[k] += beta * p[k];
    }
    if (sizeof(T) == 4 && a.fixed_bits) fixed_round24(v, a.fixed_bits);
    if (live) store24<T>(a.p, gs, s, LS, v);
    if (sizeof(T) == 2) {  // the operator must act on the stored (rounded) p
#pragma unroll
      for (int k = 0; k < 24; k++) v[k] = (C)__half2float(__float2half_rn((float)v[k]));
    }
  }
  C* slab_j = slab + j * SM::SSTRIDE;
#pragma unroll
  for (int k = 0; k < 24; k++) slab_j[k * LS + s] = v[k];
  __syncthreads();
  const int sm1 = (s == 0) ? LS - 1 : s - 1, sp1 = (s == LS - 1) ? 0 : s + 1;
  const C wm = (s == 0) ? -a.mf : (C)1, wp = (s == LS - 1) ? -a.mf : (C)1;
  C o[24];
#pragma unroll
  for (int k = 0; k < 12; k++) o[k] = a.diag * v[k] + a.off * wm * slab_j[k * LS + sm1];       // P+: psi_{s-1}
#pragma unroll
  for (int k = 12; k < 24; k++) o[k] = a.diag * v[k] + a.off * wp * slab_j[k * LS + sp1];      // P-: psi_{s+1}
  if (live) store24<T>(a.t, gs, s, LS, o);
}

// --------------------------------------------------------------------------------- BLAS-1
// One thread per (site, s) = 24 reals, runtime Ls (the chunking of the slab layout depends on the storage type, so
// mixed-precision kernels cannot treat vectors as flat arrays).  grid = (ceil(n_sites*Ls / blockDim), nblk).
struct SiteThread { long gsite; int s; bool live; int blk; };
__device__ __forceinline__ SiteThread site_thread(long n_sites, int Ls) {
  SiteThread t;
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  t.blk = blockIdx.y;
  t.live = idx < n_sites * Ls;
  const long site = t.live ? idx / Ls : 0;
  t.s = t.live ? (int)(idx - site * Ls) : 0;
  t.gsite = (long)t.blk * n_sites + site;
  return t;
}
__device__ __forceinline__ double blk_scale(const float* scale, int blk) {
  if (!scale) return 1.0;
  float sc = scale[blk];
  return sc > 0.f ? (double)sc : 1.0;
}
template <typename C> __device__ __forceinline__ C round_store(C v, int bytes) {
  return bytes == 2 ? (C)__half2float(__float2half_rn((float)v)) : v;
}

// b = a * factor * (scale[blk] or 1/scale[blk]) with precision change.
template <typename TA, typename TB>
__global__ void k_convert(const TA* __restrict__ a, TB* __restrict__ b, long n_sites, int Ls, const float* scale, int invert, double factor) {
  const SiteThread t = site_thread(n_sites, Ls);
  if (!t.live) return;
  double f = factor;
  if (scale) { const double sc = blk_scale(scale, t.blk); f *= invert ? 1.0 / sc : sc; }
  typedef typename std::conditional<(sizeof(typename ST<TA>::C) == 8 || sizeof(typename ST<TB>::C) == 8), double, float>::type A;   // no fp64 detour between fp32 / fp16 types (XU pipe)
  const A fa = (A)f;
  typename ST<TA>::C va[24]; typename ST<TB>::C vb[24];
  load24<TA>(a, t.gsite, t.s, Ls, va);
#pragma unroll
  for (int k = 0; k < 24; k++) vb[k] = (typename ST<TB>::C)((A)va[k] * fa);
  store24<TB>(b, t.gsite, t.s, Ls, vb);
}

// per-block max |a_i| (fp16 range management; reading R14).  out[blk] as float bits, atomicMax.
template <typename T>
__global__ void k_maxabs(const T* __restrict__ a, long n_sites, int Ls, float* out) {
  const SiteThread t = site_thread(n_sites, Ls);
  float m = 0.f;
  if (t.live) {
    typename ST<T>::C v[24];
    load24<T>(a, t.gsite, t.s, Ls, v);
#pragma unroll
    for (int k = 0; k < 24; k++) m = fmaxf(m, fabsf((float)v[k]));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(reinterpret_cast<unsigned int*>(out) + t.blk, __float_as_uint(m));
}

// Preconditioner prologue: r = r_in / scale[blk] stored in T;  rho0[blk] += |r|^2 of the STORED values.
template <typename TIO, typename T>
__global__ void k_pre_begin(const TIO* __restrict__ rin, T* __restrict__ r, long n_sites, int Ls, const float* scale, double* rho0, int fixed_bits = 0) {
  typedef typename ST<TIO>::C AI;   // arithmetic in the wider of the two register types: fp32 <-> fp64 conversions run on the XU pipe (16 per clock and SM)
  typedef typename ST<T>::C CT;
  __shared__ double red[32];
  const SiteThread t = site_thread(n_sites, Ls);
  double part = 0;
  if (t.live) {
    const AI f = (AI)(1.0 / blk_scale(scale, t.blk));
    AI va[24]; CT vb[24];
    load24<TIO>(rin, t.gsite, t.s, Ls, va);
#pragma unroll
    for (int k = 0; k < 24; k++) vb[k] = round_store((CT)(va[k] * f), (int)sizeof(T));
    if (sizeof(T) == 4 && fixed_bits) fixed_round24(vb, fixed_bits);
    CT acc = 0;
#pragma unroll
    for (int k = 0; k < 24; k++) acc += vb[k] * vb[k];
    part = (double)acc;
    store24<T>(r, t.gsite, t.s, Ls, vb);
  }
  const double tot = block_sum(part, red, threadIdx.x, blockDim.x);
  if (threadIdx.x == 0 && tot != 0.0) atomicAdd(rho0 + t.blk, tot);
}

// Inner-CG update of iteration `it` (reading R13):  alpha = rho[it]/pq[it] (0 once the block has stopped);
//   x += alpha p (x = alpha p at it = 0);  r -= alpha q;  rho[it+1] += |r|^2.
// last != 0: instead write z = scale * (x + alpha p) in the I/O precision and leave r alone.
template <typename T, typename TX, typename TIO>
__global__ void k_inner_update(const T* __restrict__ p, const T* __restrict__ q, T* __restrict__ r, TX* __restrict__ x,
                               TIO* __restrict__ z, long n_sites, int Ls, int it, int nblk, int last,
                               double* rho, const double* pq, const float* scale, int fixed_bits = 0) {
  typedef typename ST<TX>::C A;     // arithmetic type: fp32 unless the storage is fp64 (the scalars stay fp64; per-element fp32 <-> fp64
  typedef typename ST<T>::C CT;     // conversions would run on the XU pipe and bound the kernel: 55 % busy against DRAM 55 % before)
  __shared__ double red[32];
  const SiteThread t = site_thread(n_sites, Ls);
  const bool ok = inner_alive(rho, pq, nblk, t.blk, it);
  const A alpha = (A)(ok ? rho[(long)it * nblk + t.blk] / pq[(long)it * nblk + t.blk] : 0.0);
  double part = 0;
  if (t.live) {
    CT vp[24]; A vx[24];
    load24<T>(p, t.gsite, t.s, Ls, vp);
    if (it > 0) load24<TX>(x, t.gsite, t.s, Ls, vx);
    else {
#pragma unroll
      for (int k = 0; k < 24; k++) vx[k] = 0;
    }
#pragma unroll
    for (int k = 0; k < 24; k++) vx[k] = vx[k] + alpha * (A)vp[k];
    if (sizeof(TX) == 4 && fixed_bits) fixed_round24(vx, fixed_bits);
    if (last) {
      const A f = (A)blk_scale(scale, t.blk);
      typename ST<TIO>::C vz[24];
#pragma unroll
      for (int k = 0; k < 24; k++) vz[k] = (typename ST<TIO>::C)(vx[k] * f);
      store24<TIO>(z, t.gsite, t.s, Ls, vz);
    } else {
      store24<TX>(x, t.gsite, t.s, Ls, vx);
      CT vq[24], vr[24];
      load24<T>(q, t.gsite, t.s, Ls, vq);
      load24<T>(r, t.gsite, t.s, Ls, vr);
#pragma unroll
      for (int k = 0; k < 24; k++) vr[k] = round_store((CT)((A)vr[k] - alpha * (A)vq[k]), (int)sizeof(T));
      if (sizeof(T) == 4 && fixed_bits) fixed_round24(vr, fixed_bits);
      A acc = 0;
#pragma unroll
      for (int k = 0; k < 24; k++) acc += (A)vr[k] * (A)vr[k];
      part = (double)acc;
      store24<T>(r, t.gsite, t.s, Ls, vr);
    }
  }
  if (!last) {
    const double tot = block_sum(part, red, threadIdx.x, blockDim.x);
    if (threadIdx.x == 0 && tot != 0.0) atomicAdd(rho + (long)(it + 1) * nblk + t.blk, tot);
  }
}

// q <- what a fixed-point store of q returns (eq. 17), and pq[blk] += Re<p, q> of the stored values: the operator output of an inner
// iteration when the preconditioner's vectors live in fixed-point storage.
template <typename T>
__global__ void k_fixed_store_dot(T* __restrict__ q, const T* __restrict__ p, long n_sites, int Ls, int bits, double* pq) {
  __shared__ double red[32];
  const SiteThread t = site_thread(n_sites, Ls);
  double part = 0;
  if (t.live) {
    typename ST<T>::C vq[24], vp[24];
    load24<T>(q, t.gsite, t.s, Ls, vq);
    load24<T>(p, t.gsite, t.s, Ls, vp);
    fixed_round24(vq, bits);
#pragma unroll
    for (int k = 0; k < 24; k++) part += (double)vp[k] * (double)vq[k];
    store24<T>(q, t.gsite, t.s, Ls, vq);
  }
  const double tot = block_sum(part, red, threadIdx.x, blockDim.x);
  if (threadIdx.x == 0 && tot != 0.0) atomicAdd(pq + t.blk, tot);
}

// The storage format itself (eq. 17): ABI vector (fp64, 24 reals per colour-spinor contiguous) <-> 24 signed integers + one fp32 scale per
// colour-spinor.  One thread per colour-spinor.  INT = int8_t (limit 127) or int16_t (limit 32767).
template <typename INT>
__global__ void k_fixed_pack(const double* __restrict__ abi, INT* __restrict__ q, float* __restrict__ scale, long ncs) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ncs) return;
  const float lim = sizeof(INT) == 1 ? 127.f : 32767.f;
  float v[24], m = 0.f;
#pragma unroll
  for (int k = 0; k < 24; k++) { v[k] = (float)abi[i * 24 + k]; m = fmaxf(m, fabsf(v[k])); }
  const float safe = m > 0.f ? m : 1.f;
#pragma unroll
  for (int k = 0; k < 24; k++) q[i * 24 + k] = m > 0.f ? (INT)__float2int_rn(__fmul_rn(__fdiv_rn(v[k], safe), lim)) : (INT)0;
  scale[i] = m;
}
template <typename INT>
__global__ void k_fixed_unpack(const INT* __restrict__ q, const float* __restrict__ scale, double* __restrict__ abi, long ncs) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ncs) return;
  const float lim = sizeof(INT) == 1 ? 127.f : 32767.f;
  const float m = scale[i];
#pragma unroll
  for (int k = 0; k < 24; k++) abi[i * 24 + k] = (double)__fmul_rn(__fdiv_rn((float)q[i * 24 + k], lim), m);
}

// ------------------------------------------------------------------ reduced-Ls transfer (generic path)
// eq. 21: [T v]_{a,m} = sum_{s,n} T[a m, s n] v_{s,n}; T is the identity in colour and 4D site.
// Tm = device copy of T_host[4*Lh][4*Ls][re,im] (fp64).  One thread per (site, a = s_hat):
//   rhat = T (rin / scale[blk]) stored in T (rounded), rho0[blk] += |rhat|^2 of the stored values.
template <typename TIO, typename T>
__global__ void k_reduce_begin(const TIO* __restrict__ rin, T* __restrict__ rhat, long n_sites, int Ls, int Lh,
                               const double* __restrict__ Tm, const float* scale, double* rho0) {
  __shared__ double red[32];
  const SiteThread t = site_thread(n_sites, Lh);
  double part = 0;
  if (t.live) {
    const double f = 1.0 / blk_scale(scale, t.blk);
    double acc[24];
#pragma unroll
    for (int k = 0; k < 24; k++) acc[k] = 0;
    for (int s = 0; s < Ls; s++) {
      typename ST<TIO>::C v[24];
      load24<TIO>(rin, t.gsite, s, Ls, v);
#pragma unroll
      for (int m = 0; m < 4; m++)
#pragma unroll
        for (int n = 0; n < 4; n++) {
          const double2 tc = *reinterpret_cast<const double2*>(Tm + (((long)(t.s * 4 + m)) * (4 * Ls) + s * 4 + n) * 2);
#pragma unroll
          for (int c = 0; c < 3; c++) {
            const double vr = (double)v[(n * 3 + c) * 2], vi = (double)v[(n * 3 + c) * 2 + 1];
            acc[(m * 3 + c) * 2] += tc.x * vr - tc.y * vi;
            acc[(m * 3 + c) * 2 + 1] += tc.x * vi + tc.y * vr;
          }
        }
    }
    typename ST<T>::C o[24];
#pragma unroll
    for (int k = 0; k < 24; k++) {
      o[k] = round_store((typename ST<T>::C)(acc[k] * f), (int)sizeof(T));
      part += (double)o[k] * (double)o[k];
    }
    store24<T>(rhat, t.gsite, t.s, Lh, o);
  }
  const double tot = block_sum(part, red, threadIdx.x, blockDim.x);
  if (threadIdx.x == 0 && tot != 0.0) atomicAdd(rho0 + t.blk, tot);
}

// z = scale[blk] * T^dag xhat + mu * rin  (eq. 20).  One thread per (site, s).
template <typename TX, typename TIO>
__global__ void k_reduce_end(const TX* __restrict__ xhat, const TIO* __restrict__ rin, TIO* __restrict__ z, long n_sites, int Ls,
                             int Lh, const double* __restrict__ Tm, const float* scale, double mu) {
  const SiteThread t = site_thread(n_sites, Ls);
  if (!t.live) return;
  const double f = blk_scale(scale, t.blk);
  double acc[24];
#pragma unroll
  for (int k = 0; k < 24; k++) acc[k] = 0;
  for (int a = 0; a < Lh; a++) {
    typename ST<TX>::C v[24];
    load24<TX>(xhat, t.gsite, a, Lh, v);
#pragma unroll
    for (int m = 0; m < 4; m++)
#pragma unroll
      for (int n = 0; n < 4; n++) {
        const double2 tc = *reinterpret_cast<const double2*>(Tm + (((long)(a * 4 + m)) * (4 * Ls) + t.s * 4 + n) * 2);
#pragma unroll
        for (int c = 0; c < 3; c++) {   // conj(T) * x
          const double vr = (double)v[(m * 3 + c) * 2], vi = (double)v[(m * 3 + c) * 2 + 1];
          acc[(n * 3 + c) * 2] += tc.x * vr + tc.y * vi;
          acc[(n * 3 + c) * 2 + 1] += tc.x * vi - tc.y * vr;
        }
      }
  }
  typename ST<TIO>::C r[24], o[24];
  load24<TIO>(rin, t.gsite, t.s, Ls, r);
#pragma unroll
  for (int k = 0; k < 24; k++) o[k] = (typename ST<TIO>::C)(f * acc[k] + mu * (double)r[k]);
  store24<TIO>(z, t.gsite, t.s, Ls, o);
}

// Training of T (eq. 22, reading R20): G[a m, s n] += sum over sites and colour of
// x[a, m, c] * conj(y[s, n, c]),  x an Ls_hat vector (TX), y an Ls vector (fp64).  One thread block per SPB sites,
// both site columns staged in shared memory, thread e owns the entries e, e + blockDim, ... of the 4Lh x 4Ls matrix.
template <typename TX>
__global__ void k_outer_T(const TX* __restrict__ x, const double* __restrict__ y, long n_sites_total, int Ls, int Lh, int spb, double* __restrict__ G) {
  extern __shared__ double osm[];
  double* xs = osm;               // [Lh][24]
  double* ys = osm + 24 * Lh;     // [Ls][24]
  const int nent = 16 * Lh * Ls;
  constexpr int MAXE = 8;         // entries per thread (16*16*16 / 512)
  double accr[MAXE], acci[MAXE];
#pragma unroll
  for (int i = 0; i < MAXE; i++) { accr[i] = 0; acci[i] = 0; }
  const long s0 = (long)blockIdx.x * spb;
  for (int j = 0; j < spb; j++) {
    const long site = s0 + j;
    if (site >= n_sites_total) break;
    __syncthreads();
    for (int l = threadIdx.x; l < Lh + Ls; l += blockDim.x) {
      if (l < Lh) { typename ST<TX>::C v[24]; load24<TX>(x, site, l, Lh, v);
#pragma unroll
        for (int k = 0; k < 24; k++) xs[l * 24 + k] = (double)v[k]; }
      else { double v[24]; load24<double>(y, site, l - Lh, Ls, v);
#pragma unroll
        for (int k = 0; k < 24; k++) ys[(l - Lh) * 24 + k] = v[k]; }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < MAXE; i++) {
      const int e = threadIdx.x + i * blockDim.x;
      if (e < nent) {
        const int row = e / (4 * Ls), col = e - row * (4 * Ls);   // row = a*4 + m, col = s*4 + n
        const double* xp = xs + (row >> 2) * 24 + (row & 3) * 6;
        const double* yp = ys + (col >> 2) * 24 + (col & 3) * 6;
#pragma unroll
        for (int c = 0; c < 3; c++) {   // x * conj(y)
          accr[i] += xp[2 * c] * yp[2 * c] + xp[2 * c + 1] * yp[2 * c + 1];
          acci[i] += xp[2 * c + 1] * yp[2 * c] - xp[2 * c] * yp[2 * c + 1];
        }
      }
    }
  }
#pragma unroll
  for (int i = 0; i < MAXE; i++) {
    const int e = threadIdx.x + i * blockDim.x;
    if (e < nent) { atomicAdd(G + 2 * e, accr[i]); atomicAdd(G + 2 * e + 1, acci[i]); }
  }
}

// Same-precision flat kernels: one thread per 16-byte chunk.
template <typename T> __device__ __forceinline__ void ldchunk(const T* base, long i, typename ST<T>::C* v) {
  typedef typename ST<T>::V V; V q = __ldg(reinterpret_cast<const V*>(base) + i); unpackV(q, v);
}
template <typename T> __device__ __forceinline__ void stchunk(T* base, long i, const typename ST<T>::C* v) {
  typedef typename ST<T>::V V; V q; packV(q, v); reinterpret_cast<V*>(base)[i] = q;
}

// Device-resident scalars of the outer iteration (Algorithm 1; eq. 18): no host round trip between the kernels.
//   sc[0] <p,Ap> (kernel 5)   sc[1] |r_{k+1}|^2   sc[2] <z_{k+1},r_{k+1}>   sc[3] <z_{k+1},A p_k>   (accumulators, zeroed by k_outer_scalars)
//   sc[4] <z_k,r_k>   sc[5] alpha_k   sc[6] beta_k   sc[7] <z,r> before the last k_outer_scalars (denominator for a redo after a replacement)
enum { SC_PAP = 0, SC_RR = 1, SC_RZN = 2, SC_ZAP = 3, SC_RZ = 4, SC_ALPHA = 5, SC_BETA = 6, SC_RZ_PREV = 7, SC_N = 8 };

// alpha = <r,z> / <p,Ap> (0 if <p,Ap> <= 0: the host reports the breakdown), x += alpha p, r -= alpha Ap, sc[SC_RR] += |r|^2.
// self_z (plain CG, z = r): also sc[SC_RZN] += |r|^2 and sc[SC_ZAP] += <r, Ap>, the two inner products of eq. 18, in the same pass.
template <typename T>
__global__ void k_outer_update(const T* __restrict__ p, const T* __restrict__ q, T* __restrict__ r, T* __restrict__ x,
                               long nchunk, double* __restrict__ sc, int self_z) {
  __shared__ double red[32];
  constexpr int PER = ST<T>::PER;
  typedef typename ST<T>::C A;      // arithmetic in the register type of the storage (fp32 for fp16 / fp32 storage): no per-element fp64 conversions (XU pipe)
  const double pq = sc[SC_PAP];
  const double alpha = pq > 0.0 ? sc[SC_RZ] / pq : 0.0;
  const A al = (A)alpha;
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  double part = 0, part2 = 0;
  if (i < nchunk) {
    A vp[PER], vq[PER], vr[PER], vx[PER];
    ldchunk<T>(p, i, vp); ldchunk<T>(q, i, vq); ldchunk<T>(r, i, vr); ldchunk<T>(x, i, vx);
    A a1 = 0, a2 = 0;
#pragma unroll
    for (int k = 0; k < PER; k++) {
      vx[k] = vx[k] + al * vp[k];
      vr[k] = round_store(vr[k] - al * vq[k], (int)sizeof(T));
      a1 += vr[k] * vr[k];
      a2 += vr[k] * vq[k];
    }
    part = (double)a1; part2 = (double)a2;
    stchunk<T>(x, i, vx); stchunk<T>(r, i, vr);
  }
  const double tot = block_sum(part, red, threadIdx.x, blockDim.x);
  __syncthreads();
  const double tot2 = self_z ? block_sum(part2, red, threadIdx.x, blockDim.x) : 0.0;
  if (threadIdx.x == 0) {
    atomicAdd(sc + SC_RR, tot);
    if (self_z) { atomicAdd(sc + SC_RZN, tot); atomicAdd(sc + SC_ZAP, tot2); }
    if (blockIdx.x == 0) sc[SC_ALPHA] = alpha;
  }
}

// End of an outer iteration, one thread: beta_k of eq. 18, <z,r> <- <z',r'>, snapshot of (<p,Ap>, |r|^2) for the
// host's lagged polling, accumulators cleared for the next iteration.
//   mode 0: beta = -alpha <z',Ap> / <z,r>     (eq. 18 with r' - r = -alpha A p)
//   mode 1: beta = <z',r'> / (f2 * <z,r>)     right after a residual replacement (Alg. 1's ratio, R16); f2 = (sigma_old/sigma_new)^2
//           rescales <z,r> to the new unit of the fp16 sloppy vectors (R17b), 1 otherwise
//   mode 2: as mode 1 but against the <z,r> saved before the previous call (the z of the replaced residual is recomputed)
//   mode 3: start: <z,r> <- <z_0,r_0>, beta = 0
__global__ void k_outer_scalars(double* __restrict__ sc, double* __restrict__ snap, int mode, double f2) {
  const double rzn = sc[SC_RZN];
  if (snap) { snap[0] = sc[SC_PAP]; snap[1] = sc[SC_RR]; }
  if (mode == 3) { sc[SC_RZ] = rzn; sc[SC_RZ_PREV] = rzn; sc[SC_BETA] = 0.0; }
  else {
    const double rz = mode == 2 ? sc[SC_RZ_PREV] : sc[SC_RZ];
    double beta;
    if (mode == 0) beta = -sc[SC_ALPHA] * sc[SC_ZAP] / rz; else beta = rzn / (f2 * rz);
    if (!(rz != 0.0)) beta = 0.0;
    if (mode != 2) sc[SC_RZ_PREV] = rz;
    sc[SC_BETA] = beta; sc[SC_RZ] = rzn;
  }
  sc[SC_PAP] = 0.0; sc[SC_RR] = 0.0; sc[SC_RZN] = 0.0; sc[SC_ZAP] = 0.0;
}

// out[0] += <a,b>, out[1] += <a,c> (c may be null): the inner products of the Polak-Ribiere beta (eq. 18, R16).
template <typename T>
__global__ void k_dot2(const T* __restrict__ a, const T* __restrict__ b, const T* __restrict__ c, long nchunk, double* out) {
  __shared__ double red[32];
  constexpr int PER = ST<T>::PER;
  double p0 = 0, p1 = 0;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nchunk; i += (long)gridDim.x * blockDim.x) {
    typename ST<T>::C va[PER], vb[PER], vc[PER];
    ldchunk<T>(a, i, va); ldchunk<T>(b, i, vb);
    if (c) ldchunk<T>(c, i, vc);
    typename ST<T>::C q0 = 0, q1 = 0;    // one chunk in the register type, then one conversion (no per-element fp64 conversions: XU pipe)
#pragma unroll
    for (int k = 0; k < PER; k++) { q0 += va[k] * vb[k]; if (c) q1 += va[k] * vc[k]; }
    p0 += (double)q0; p1 += (double)q1;
  }
  const double t0 = block_sum(p0, red, threadIdx.x, blockDim.x);
  __syncthreads();
  const double t1 = block_sum(p1, red, threadIdx.x, blockDim.x);
  if (threadIdx.x == 0) { atomicAdd(out, t0); if (c) atomicAdd(out + 1, t1); }
}

// y = a*x + b*y elementwise, coefficients by value (fp64 bookkeeping of the reliable updates, R17).
template <typename T>
__global__ void k_axpby(double a, const T* __restrict__ x, double b, T* __restrict__ y, long nchunk) {
  constexpr int PER = ST<T>::PER;
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nchunk) return;
  typename ST<T>::C vx[PER], vy[PER];
  ldchunk<T>(x, i, vx); ldchunk<T>(y, i, vy);
#pragma unroll
  for (int k = 0; k < PER; k++) vy[k] = (typename ST<T>::C)a * vx[k] + (typename ST<T>::C)b * vy[k];
  stchunk<T>(y, i, vy);
}

// -------------------------------------------------------------------------------- layout conversion and gauge ingest
// ABI psi[s][x_cb][24] (fp64; fp32 for the *_host32 entry points)  <->  native v[i][chunk][s][PER] (i = FULL E-list index), SURVEY 8(b).
template <typename T, int LS, typename TA>
__global__ void k_pack(const TA* __restrict__ abi, T* __restrict__ nat, const int* __restrict__ int_to_cb, long Vh, int to_native) {
  typedef typename ST<T>::C C;
  const long i = (long)blockIdx.x * Tile<LS>::NS + threadIdx.y;
  const int s = threadIdx.x;
  if (i >= Vh) return;
  const long cb = int_to_cb[i];
  TA* a = const_cast<TA*>(abi) + ((long)s * Vh + cb) * 24;
  C v[24];
  if (to_native) {
#pragma unroll
    for (int k = 0; k < 24; k++) v[k] = (C)a[k];
    store24<T>(nat, i, s, LS, v);
  } else {
    load24<T>(nat, i, s, LS, v);
#pragma unroll
    for (int k = 0; k < 24; k++) a[k] = (TA)v[k];
  }
}

__device__ __forceinline__ void st_link_real(double* p, double v) { *p = v; }
__device__ __forceinline__ void st_link_real(float* p, double v) { *p = (float)v; }
__device__ __forceinline__ void st_link_real(__half* p, double v) { *p = __float2half_rn((float)v); }

// Per-stage link copies: for list site i of block blk and dir = 2*mu+bw:
//   bw = 0: W = U_mu(x);  bw = 1: W = U_mu(x - mu)^dag;  x = (origin(blk) + c_i) mod L, the GLOBAL periodic index
// (reading R10: pad sites read links by global periodic index).  flip bit d set  <=>  the link crosses the
// antiperiodic time boundary (R7); with ng = 18 the sign is folded into the stored link instead and the bit stays clear.
// Stored: first ng reals of W (ng = 12: two rows, R8).
template <typename T>
__global__ void k_build_links(const double* __restrict__ U_abi, T* __restrict__ links, uint8_t* __restrict__ flip,
                              const short* __restrict__ coords, const short* __restrict__ origin, long n_list, int nblk,
                              int Lx, int Ly, int Lz, int Lt, int tb, int ng) {
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long)nblk * n_list) return;
  const int blk = (int)(idx / n_list);
  const long i = idx % n_list;
  const int L[4] = {Lx, Ly, Lz, Lt};
  const long Vh = (long)Lx * Ly * Lz * Lt / 2;
  int x[4];
#pragma unroll
  for (int d = 0; d < 4; d++) { int v = ((int)origin[4 * blk + d] + (int)coords[4 * i + d]) % L[d]; x[d] = v < 0 ? v + L[d] : v; }
  unsigned fl = 0;
  for (int mu = 0; mu < 4; mu++)
    for (int bw = 0; bw < 2; bw++) {
      int y[4] = {x[0], x[1], x[2], x[3]};
      if (bw) y[mu] = (y[mu] + L[mu] - 1) % L[mu];
      const int par = (y[0] + y[1] + y[2] + y[3]) & 1;
      const long lex = y[0] + (long)Lx * (y[1] + (long)Ly * (y[2] + (long)Lz * y[3]));
      const double* u = U_abi + (((long)mu * 2 + par) * Vh + lex / 2) * 18;
      // 18 stored reals: the sign is folded into the link; 12 reals: it must be applied after the third row is rebuilt (R7, R8)
      double sgn = 1.0;
      if (mu == 3 && tb == -1 && y[3] == Lt - 1) { if (ng == 18) sgn = -1.0; else fl |= 1u << (2 * mu + bw); }
      T* g = links + (idx * 8 + 2 * mu + bw) * ng;
      for (int q = 0; q < ng / 2; q++) {
        const int r = q / 3, c = q % 3;
        double re, im;
        if (!bw) { re = u[(r * 3 + c) * 2]; im = u[(r * 3 + c) * 2 + 1]; }
        else     { re = u[(c * 3 + r) * 2]; im = -u[(c * 3 + r) * 2 + 1]; }
        st_link_real(g + 2 * q, sgn * re); st_link_real(g + 2 * q + 1, sgn * im);
      }
    }
  flip[idx] = (uint8_t)fl;
}

}  // namespace mspcg
#include "transfer_tc.cuh"
#include "dense5d_tma.cuh"
