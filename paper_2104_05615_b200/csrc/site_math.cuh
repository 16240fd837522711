// site_math.cuh -- per-site arithmetic of the Wilson hop (eq. 8) in the chiral basis of reading R2:
//   gamma_k = [[0, -i sigma_k], [+i sigma_k, 0]] (k = x,y,z),  gamma_4 = [[0, 1], [1, 0]],  gamma5 = diag(+,+,-,-).
// A spinor is 24 reals, index (spin*3 + colour)*2 + reim.  A link is 18 reals, index (row*3 + col)*2 + reim.
//
// One hop term is  (1 + sigma * gamma_mu) W psi  with W the 3x3 colour matrix (U_mu(x) for the forward neighbour,
// U_mu(x-mu)^dag -- stored already daggered -- for the backward one) and sigma = -1 forward / +1 backward, both
// negated for D^w^dag (gamma_mu -> -gamma_mu, reading R6).  With psi = (u, l) the upper / lower two spin components:
//   spatial k: (1 + sigma g_k) psi = (h, sigma i sigma_k h),  h = u - sigma i sigma_k l
//   time     : (1 + sigma g_4) psi = (h, sigma h),            h = u + sigma l
// so only the half spinor h (2 spins x 3 colours) is multiplied by W (the "SU(3) link x half-spinor" of PAPER.md:220).
#pragma once

#if defined(__CUDACC__)
#define MSPCG_HD __host__ __device__ __forceinline__
#else
#define MSPCG_HD inline
#endif

namespace mspcg {

// chi[2][3] (complex) = W * h[2][3]: 2 x (3x3 complex matrix times 3-vector)
template <typename C>
MSPCG_HD void su3_mul_half(C chi[12], const C W[18], const C h[12]) {
#pragma unroll
  for (int sp = 0; sp < 2; sp++)
#pragma unroll
    for (int r = 0; r < 3; r++) {
      C re = 0, im = 0;
#pragma unroll
      for (int c = 0; c < 3; c++) {
        C wr = W[(r * 3 + c) * 2], wi = W[(r * 3 + c) * 2 + 1];
        C hr = h[(sp * 3 + c) * 2], hi = h[(sp * 3 + c) * 2 + 1];
        re += wr * hr; re -= wi * hi;
        im += wr * hi; im += wi * hr;
      }
      chi[(sp * 3 + r) * 2] = re; chi[(sp * 3 + r) * 2 + 1] = im;
    }
}

// acc += (1 + sigma*gamma_mu) W psi.   MU is a compile-time direction 0..3 (x,y,z,t).
template <int MU, typename C>
MSPCG_HD void hop_term(C acc[24], const C psi[24], const C W[18], C sigma) {
  C h[12], chi[12];
  // spin s, colour c, re/im -> psi[(s*3+c)*2 + ri];  u = spins 0,1;  l = spins 2,3
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const C u0r = psi[(0 * 3 + c) * 2], u0i = psi[(0 * 3 + c) * 2 + 1];
    const C u1r = psi[(1 * 3 + c) * 2], u1i = psi[(1 * 3 + c) * 2 + 1];
    const C l0r = psi[(2 * 3 + c) * 2], l0i = psi[(2 * 3 + c) * 2 + 1];
    const C l1r = psi[(3 * 3 + c) * 2], l1i = psi[(3 * 3 + c) * 2 + 1];
    if (MU == 0) {        // i sigma_1 (a,b) = (i b, i a):  h0 = u0 - sigma i l1,  h1 = u1 - sigma i l0
      h[(0 * 3 + c) * 2] = u0r + sigma * l1i; h[(0 * 3 + c) * 2 + 1] = u0i - sigma * l1r;
      h[(1 * 3 + c) * 2] = u1r + sigma * l0i; h[(1 * 3 + c) * 2 + 1] = u1i - sigma * l0r;
    } else if (MU == 1) { // i sigma_2 (a,b) = (b, -a):     h0 = u0 - sigma l1,    h1 = u1 + sigma l0
      h[(0 * 3 + c) * 2] = u0r - sigma * l1r; h[(0 * 3 + c) * 2 + 1] = u0i - sigma * l1i;
      h[(1 * 3 + c) * 2] = u1r + sigma * l0r; h[(1 * 3 + c) * 2 + 1] = u1i + sigma * l0i;
    } else if (MU == 2) { // i sigma_3 (a,b) = (i a, -i b): h0 = u0 - sigma i l0,  h1 = u1 + sigma i l1
      h[(0 * 3 + c) * 2] = u0r + sigma * l0i; h[(0 * 3 + c) * 2 + 1] = u0i - sigma * l0r;
      h[(1 * 3 + c) * 2] = u1r - sigma * l1i; h[(1 * 3 + c) * 2 + 1] = u1i + sigma * l1r;
    } else {              // time: h = u + sigma l
      h[(0 * 3 + c) * 2] = u0r + sigma * l0r; h[(0 * 3 + c) * 2 + 1] = u0i + sigma * l0i;
      h[(1 * 3 + c) * 2] = u1r + sigma * l1r; h[(1 * 3 + c) * 2 + 1] = u1i + sigma * l1i;
    }
  }
  su3_mul_half(chi, W, h);
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const C x0r = chi[(0 * 3 + c) * 2], x0i = chi[(0 * 3 + c) * 2 + 1];
    const C x1r = chi[(1 * 3 + c) * 2], x1i = chi[(1 * 3 + c) * 2 + 1];
    acc[(0 * 3 + c) * 2] += x0r; acc[(0 * 3 + c) * 2 + 1] += x0i;
    acc[(1 * 3 + c) * 2] += x1r; acc[(1 * 3 + c) * 2 + 1] += x1i;
    if (MU == 0) {        // lower = sigma (i x1, i x0)
      acc[(2 * 3 + c) * 2] -= sigma * x1i; acc[(2 * 3 + c) * 2 + 1] += sigma * x1r;
      acc[(3 * 3 + c) * 2] -= sigma * x0i; acc[(3 * 3 + c) * 2 + 1] += sigma * x0r;
    } else if (MU == 1) { // lower = sigma (x1, -x0)
      acc[(2 * 3 + c) * 2] += sigma * x1r; acc[(2 * 3 + c) * 2 + 1] += sigma * x1i;
      acc[(3 * 3 + c) * 2] -= sigma * x0r; acc[(3 * 3 + c) * 2 + 1] -= sigma * x0i;
    } else if (MU == 2) { // lower = sigma (i x0, -i x1)
      acc[(2 * 3 + c) * 2] -= sigma * x0i; acc[(2 * 3 + c) * 2 + 1] += sigma * x0r;
      acc[(3 * 3 + c) * 2] += sigma * x1i; acc[(3 * 3 + c) * 2 + 1] -= sigma * x1r;
    } else {              // lower = sigma (x0, x1)
      acc[(2 * 3 + c) * 2] += sigma * x0r; acc[(2 * 3 + c) * 2 + 1] += sigma * x0i;
      acc[(3 * 3 + c) * 2] += sigma * x1r; acc[(3 * 3 + c) * 2 + 1] += sigma * x1i;
    }
  }
}

// Third row of an SU(3) matrix from its first two (reading R8): row2 = conj(row0 x row1).
template <typename C>
MSPCG_HD void su3_third_row(C W[18]) {
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
    // (row0 x row1)_c = a_{c1} b_{c2} - a_{c2} b_{c1}
    C ar = W[c1 * 2], ai = W[c1 * 2 + 1], br = W[(3 + c2) * 2], bi = W[(3 + c2) * 2 + 1];
    C cr = W[c2 * 2], ci = W[c2 * 2 + 1], dr = W[(3 + c1) * 2], di = W[(3 + c1) * 2 + 1];
    C re = (ar * br - ai * bi) - (cr * dr - ci * di);
    C im = (ar * bi + ai * br) - (cr * di + ci * dr);
    W[(6 + c) * 2] = re; W[(6 + c) * 2 + 1] = -im;
  }
}

}  // namespace mspcg
