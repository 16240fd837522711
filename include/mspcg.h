/* mspcg.h -- C ABI of libmspcg: the single-GPU (B200, sm_100a) hot path of multi-splitting preconditioned CG
 * (MSPCG) for the even-odd preconditioned Moebius domain-wall normal equations  D^dag D x = b.
 *
 * Paper: arXiv 2104.05615 (PAPER.md in the reference mount).  Citations below are PAPER.md line numbers plus the
 * section / equation; "R<n>" are the readings of silent or garbled passages listed in DESIGN.md.
 *
 * Plain C, plain pointers and sizes.  Every pointer says whether it is HOST or DEVICE memory.  The library never
 * allocates device memory for vectors, tables or link copies: the caller (PyTorch, in this repository) owns one
 * workspace buffer and every input / output buffer.  All calls return an mspcg status (0 = OK, negative = error),
 * never throw and never exit; mspcg_last_error() gives a message for the last failing call on that context.
 *
 * ---------------------------------------------------------------------------------------------------------------
 * Vector layouts
 *
 *  ABI layout (fp64 only): even-parity 5D spinor  psi[s][x_cb][spin 4][colour 3][re,im],  x_cb = lex/2 over even
 *      sites, lex = x + Lx*(y + Ly*(z + Lz*t)), parity = (x+y+z+t) mod 2 (eq. 3).  Spin index in the
 *      chiral basis of R2 (gamma5 = diag(+,+,-,-)).  Ls*V4/2*24 doubles.
 *  NATIVE layout (precision prec): the library's private site-slab layout, mspcg_vec_bytes(ctx, prec) bytes; made by
 *      mspcg_pack and read back by mspcg_unpack.  Operator calls on NATIVE vectors do no layout conversion.
 *  Gauge ABI layout: U[mu][parity][x_cb][row 3][col 3][re,im] fp64, mu = 0..3 <-> x,y,z,t, periodic links (the
 *      antiperiodic time boundary is requested with t_boundary = -1 and folded in by the library, R7).
 * --------------------------------------------------------------------------------------------------------------- */
#ifndef MSPCG_H
#define MSPCG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mspcg_ctx mspcg_ctx; /* opaque, library-owned (host memory) */

enum { MSPCG_OK = 0, MSPCG_EINVAL = -1, MSPCG_ENOMEM = -2, MSPCG_ECUDA = -3, MSPCG_ENOGAUGE = -4,
       MSPCG_ENOCONV = -5, MSPCG_EBREAKDOWN = -6, MSPCG_ENOWORKSPACE = -7 };
enum { MSPCG_F64 = 8, MSPCG_F32 = 4, MSPCG_F16 = 2 };   /* storage precision of vectors and link copies       */
enum { MSPCG_LAYOUT_ABI = 0, MSPCG_LAYOUT_NATIVE = 1 }; /* layout of the in/out buffers of the apply calls    */

/* Create a context: lattice Lx,Ly,Lz,Lt (all even), fifth dimension Ls, Moebius parameters b, c, M5 (domain-wall
 * height) and mf (eq. 4-8; operator entries: R1-R4), and the Dirichlet block ("virtual node",
 * PAPER.md:162-176 eq. 12-14) extents Bx..Bt: every B even, dividing L; B == L means that direction is not cut.
 * HOST-only work (index tables, Ls x Ls matrices): needs no GPU.  Errors: MSPCG_EINVAL for odd L or B, L % B != 0,
 * Ls < 2 or not one of the compiled values {4,6,8,12,16}, alpha = b(4-M5)+1 == 0. */
int mspcg_create(mspcg_ctx** out, int Lx, int Ly, int Lz, int Lt, int Ls, double b, double c, double M5, double mf,
                 int Bx, int By, int Bz, int Bt);
int mspcg_destroy(mspcg_ctx* ctx);
const char* mspcg_last_error(const mspcg_ctx* ctx);

/* Host-side geometry facts (no GPU): out[0]=number of blocks, out[1]=4D sites of one parity inside a block (E0),
 * out[2]=even 4D sites with L1 overshoot <= 2 (E2), out[3]=odd 4D sites with overshoot <= 1 (O1)
 * (minimal site sets of PAPER.md:226, R11), out[4]=V4/2. */
int mspcg_geometry(const mspcg_ctx* ctx, long out[5]);
/* The P+ chirality block (Ls x Ls, row major, HOST) of which = 0: M5, 1: Mphi, 2: M5^-1 (R3, R4). */
int mspcg_get_matrix(const mspcg_ctx* ctx, int which, double* out_host);

/* Precisions this context will run in, and the workspace they need.  outer_prec: the sloppy precision of the outer
 * iteration and of mspcg_apply_MdagM besides fp64 (fp64 is always available); inner_prec: storage precision of the
 * preconditioner (R14); recon: 18, or 12 = two-row link storage with the third row rebuilt in the
 * kernels (R8) for the non-fp64 link copies.  Returns the byte count through *bytes. */
int mspcg_workspace_bytes(mspcg_ctx* ctx, int outer_prec, int inner_prec, int recon, size_t* bytes);
/* Hand the library its workspace (DEVICE, 256-byte aligned, >= the size above; caller keeps ownership and must keep
 * it alive until mspcg_destroy).  Uploads the index tables on `stream` (a cudaStream_t passed as void*). */
int mspcg_set_workspace(mspcg_ctx* ctx, void* workspace_dev, size_t bytes, void* stream);

/* Ingest a gauge field: U_dev is DEVICE fp64 in the gauge ABI layout (4*V4*18
 * doubles).  t_boundary = +1 periodic / -1 antiperiodic in time (R7).  Builds the per-stage link copies in every
 * configured precision.  Asynchronous on `stream`. */
int mspcg_load_gauge(mspcg_ctx* ctx, const double* U_dev, int t_boundary, void* stream);

/* NATIVE <-> ABI conversion of even-parity vectors (DEVICE pointers, asynchronous). */
size_t mspcg_vec_bytes(const mspcg_ctx* ctx, int prec);
int mspcg_pack(mspcg_ctx* ctx, const double* abi_dev, void* native_dev, int prec, void* stream);
int mspcg_unpack(mspcg_ctx* ctx, const void* native_dev, double* abi_dev, int prec, void* stream);

/* out = M5^-1 in (dagger = 0) or M5^-dag in (dagger != 0) on an fp16 NATIVE one-parity vector (mspcg_pack with MSPCG_F16):
 * the dense fifth-dimension contraction of PAPER.md:260-264 (an Ls x Ls real matrix per chirality times the Ls x 24*sites
 * panel; M5^-1 of eq. 4-5, closed form R4) as a stand-alone tcgen05.mma GEMM with fp16 operands and fp32
 * accumulation in tensor memory.  Inside mspcg_apply_MdagM / mspcg_apply_precond the same contraction is fused into the
 * hop kernels; this entry point applies it on its own.  Ls must be 8, 12 or 16.  in_dev, out_dev: DEVICE, caller-owned,
 * mspcg_vec_bytes(ctx, MSPCG_F16) bytes each, must not alias.  Needs the workspace, not the gauge field.  Asynchronous
 * on `stream`.  Errors: ENOWORKSPACE, EINVAL, ECUDA. */
int mspcg_apply_M5inv(mspcg_ctx* ctx, const void* in_dev, void* out_dev, int dagger, void* stream);

/* out = D^dag D in  on the whole periodic/antiperiodic lattice (eq. 9-10, 230-258 eq. 15-16:
 * one Mphi kernel and four fused hop kernels).  prec = MSPCG_F64 or the configured outer_prec.
 * layout ABI: in/out are fp64 ABI vectors (converted on entry/exit); NATIVE: vectors of `prec` from mspcg_pack.
 * in and out must not alias.  Asynchronous on `stream`.  Errors: ENOGAUGE, ENOWORKSPACE, EINVAL. */
int mspcg_apply_MdagM(mspcg_ctx* ctx, const void* in_dev, void* out_dev, int prec, int layout, void* stream);

/* z = M^-1 r: the multi-splitting preconditioner (eq. 12-14): for every Dirichlet block
 * independently, n_inner CG iterations from a zero guess (R13) on A_s z_s = r_s, A_s being the block's
 * part of D^dag D including the snake terms (eq. 11, 224-228; R10 reading PAD).  All blocks run
 * batched in the same launches.  io_prec: precision of r and z (F64 or outer_prec); the inner iteration runs in the
 * configured inner_prec (fp16 storage: per-block max-abs scaling, fp32 arithmetic).  If a reduced-Ls transfer
 * matrix is set and use_reduced != 0:  z = T^dag CG_k[M-hat](T r) + mu r (eq. 19-21). */
int mspcg_apply_precond(mspcg_ctx* ctx, const void* r_dev, void* z_dev, int io_prec, int layout, int n_inner,
                        int use_reduced, void* stream);
/* The same two operator calls on HOST fp64 ABI buffers: host->device copy, apply, device->host copy, synchronous.
 * (End-to-end path used by bench.py's e2e figure.) */
int mspcg_apply_MdagM_host(mspcg_ctx* ctx, const double* in_host, double* out_host, int prec);
int mspcg_apply_precond_host(mspcg_ctx* ctx, const double* r_host, double* z_host, int io_prec, int n_inner,
                             int use_reduced);

/* The same with SINGLE-precision host vectors (ABI layout psi[s][x_cb][4][3][re,im] in float, HOST, pinned for full PCIe speed): half the
 * PCIe bytes for computations that run in fp32 or fp16 anyway.  prec / io_prec: MSPCG_F32 or MSPCG_F16 (MSPCG_EINVAL for fp64).  Synchronous. */
int mspcg_apply_MdagM_host32(mspcg_ctx* ctx, const float* in_host, float* out_host, int prec);
int mspcg_apply_precond_host32(mspcg_ctx* ctx, const float* r_host, float* z_host, int io_prec, int n_inner, int use_reduced);

/* A_s applied to the block-`block` part of a vector (debug / parity entry: PAPER.md:224, R10): fp64, ABI layout;
 * out is zero outside the block. */
int mspcg_apply_A_block(mspcg_ctx* ctx, const double* in_dev, double* out_dev, int block, int prec, void* stream);

/* Full 4-step solve: the set-up and tear-down around mspcg_solve for the unpreconditioned system of
 * PAPER.md:91 eq. (4), [[M5, M4eo],[M4oe, M5]] (psi_e, psi_o) = (phi_e, phi_o).  All vectors DEVICE fp64, ABI layout; an
 * ODD-parity vector is psi[s][x_cb][4][3][re,im] with x_cb = lex(x,y,z,t; x fastest)/2 over the odd sites.  fp64 arithmetic.
 *   mspcg_prepare_source:  phihat_e = M5^-1 phi_e - M5^-1 M4eo M5^-1 phi_o (eq. 6) -> phihat_e_dev (or NULL),
 *                          rhs = D^dag phihat_e (eq. 9) -> rhs_dev, the `b` of mspcg_solve;
 *   mspcg_reconstruct_odd: psi_o = M5^-1 (phi_o - M4oe psi_e) (second row of eq. 4) from the solution psi_e of mspcg_solve;
 *   mspcg_apply_full:      (out_e, out_o) = the 2x2 operator of eq. (4) applied to (psi_e, psi_o), to check a solution.
 * They use the solver's vectors as scratch (do not run concurrently with mspcg_solve on another stream).  Outputs may not
 * alias inputs.  Errors: MSPCG_EINVAL (null pointer), MSPCG_ENOGAUGE / MSPCG_ENOWORKSPACE, MSPCG_ECUDA. */
int mspcg_prepare_source(mspcg_ctx* ctx, const double* phi_e_dev, const double* phi_o_dev, double* phihat_e_dev, double* rhs_dev, void* stream);
int mspcg_reconstruct_odd(mspcg_ctx* ctx, const double* psi_e_dev, const double* phi_o_dev, double* psi_o_dev, void* stream);
int mspcg_apply_full(mspcg_ctx* ctx, const double* psi_e_dev, const double* psi_o_dev, double* out_e_dev, double* out_o_dev, void* stream);

/* Reduced-Ls preconditioner: Ls_hat in {4,6,8,12,16}, Ls_hat <= Ls; T_host[4*Ls_hat][4*Ls][re,im]
 * (HOST, copied; row (s_hat,spin), column (s,spin); identity in colour and 4D site, eq. 21), shift mu (eq. 20).  The
 * reduced operator uses the same b, c, M5, mf (reading R19).  Must be called before mspcg_workspace_bytes.  Afterwards
 * use_reduced != 0 in mspcg_apply_precond / use_reduced_ls in mspcg_solve_params selects
 *     z = T^dag CG_k[Mhat](T r) + mu r ;
 * the full-Ls preconditioner of the same context stays available.  With fp16 inner storage and (Ls, Ls_hat) in
 * {(8,4),(12,6),(12,8),(16,8),(16,12)} the two transfers run as tcgen05.mma contractions (fp16 operands, fp32
 * accumulation), otherwise on the CUDA cores in fp64.  Errors: MSPCG_EINVAL (bad Ls_hat, null T, called too late). */
int mspcg_set_reduced_ls(mspcg_ctx* ctx, int Ls_hat, const double* T_host, double mu);

/* Replace T and mu of a context whose workspace is already set (HOST T as in mspcg_set_reduced_ls, same Ls_hat). */
int mspcg_update_T(mspcg_ctx* ctx, const double* T_host, double mu, void* stream);

/* Training of T (eq. 22; reading R20) -- a set-up step, not on the timed path.
 *   chi2 = sum_i | M (T^dag Ahat T + mu) v_i - v_i |^2 ,   M = (+)_s A_s (full Ls),  Ahat = n_inner block-CG steps at Ls_hat,
 *   grad = d chi2 / d conj(T) = sum_i (c_i v_i^dag + a_i g_i^dag)  with Ahat treated as a fixed Hermitian operator
 *   (e = M w - v, g = M e, a = Ahat T v, c = Ahat T g), layout of T_host.
 * v_dev: nvec DEVICE fp64 ABI vectors, contiguous (the paper uses residual vectors of a full-Ls MSPCG run).  chi2_host:
 * HOST double; grad_host: HOST [4*Ls_hat][4*Ls][re,im] or NULL.  Needs inner_prec fp64 or fp32 (EINVAL for fp16: train in
 * one context, use T in any).  Synchronous. */
int mspcg_train_eval(mspcg_ctx* ctx, const double* v_dev, int nvec, int n_inner, double* chi2_host, double* grad_host, void* stream);
/* n_steps of: P = -grad + momentum * P_prev; chi2 at eta0 * (0, 1/2, 1, 3/2, 2), eta0 = chi2 / |grad|^2; T += eta* P with eta*
 * the minimiser over [0, 2 eta0] of the quartic through the five values ("line search", "momentum method"), kept
 * only if the loss there is not above the best sampled value; a step without decrease drops the momentum and quarters eta0.
 * The context's T
 * is updated; T_host_out (HOST, layout of T_host) receives it; chi2_history_host (HOST, n_steps + 1 doubles or NULL) the
 * loss before every step and after the last. */
int mspcg_train_T(mspcg_ctx* ctx, const double* v_dev, int nvec, int n_inner, int n_steps, double momentum, double* T_host_out,
                  double* chi2_history_host, void* stream);

typedef struct {
  double tol;          /* relative residual |r|/|b| (R15)                                                        */
  int max_iter;        /* outer iteration cap                                                                    */
  int use_precond;     /* 0: plain CG (z = r), 1: MSPCG                                                          */
  int n_inner;         /* inner CG iterations per block                                           */
  int sloppy_prec;     /* MSPCG_F64 (no reliable updates needed) or the configured outer_prec                    */
  double delta;        /* reliable-update threshold (R17), e.g. 0.1                                              */
  int use_reduced_ls;  /* 0/1                                                                                    */
  int history_len;     /* entries available in `history` (HOST) or 0                                             */
  double* history;     /* HOST: |r_k|/|b| of the iterated residual for k = 1..                                   */
} mspcg_solve_params;

typedef struct {
  int iters, reliable_updates, converged, breakdown;
  long inner_applies;  /* total A_s applications (blocks x inner iterations x outer applications)                */
  long outer_applies;  /* D^dag D applications, sloppy + precise                                                 */
  double true_res;     /* |b - A x| / |b| in fp64                                                                */
  double seconds;      /* device time of the solve, CUDA events                                                  */
} mspcg_solve_stats;

/* Solve D^dag D x = b (eq. 9) with Algorithm 1 (R15), Polak-Ribiere beta
 * (eq. 18; R16) and reliable updates (R17).  b_dev, x_dev: DEVICE fp64 ABI vectors;
 * x_dev holds x0 on entry and the solution on exit.  Synchronous: returns when *stats (HOST) is valid.
 * Returns MSPCG_OK, MSPCG_ENOCONV (max_iter hit, x = best iterate) or MSPCG_EBREAKDOWN (<p,Ap> <= 0 or NaN). */
int mspcg_solve(mspcg_ctx* ctx, const double* b_dev, double* x_dev, const mspcg_solve_params* params,
                mspcg_solve_stats* stats, void* stream);

/* r = b - D^dag D x in fp64 (the true residual of PAPER.md:117 eq. 9; the training vectors of PAPER.md:322 are such residuals of
 * a full-Ls MSPCG run).  b_dev, x_dev, r_dev: DEVICE fp64 ABI vectors; r_dev may not alias b_dev or x_dev.  normalise != 0:
 * r is divided by |r|_2 (left as is when r = 0).  *rnorm_host (HOST, may be NULL) receives |b - D^dag D x|_2.  Synchronous.
 * Uses the solver's vectors as scratch.  Errors: MSPCG_EINVAL (null pointer, aliasing), MSPCG_ENOGAUGE / MSPCG_ENOWORKSPACE. */
int mspcg_residual(mspcg_ctx* ctx, const double* b_dev, const double* x_dev, double* r_dev, int normalise, double* rnorm_host,
                   void* stream);

/* Block-resident inner CG (preconditioner kernels are global-memory or L2 bound; blocks are
 * independent).  blocks_per_group = G > 0: mspcg_apply_precond (and the preconditioner inside mspcg_solve) runs all inner iterations for G
 * Dirichlet blocks at a time, reusing the same G-block buffers for every group, so that with G x (per-block working set) below the
 * 126 MB L2 the inner vectors never travel to HBM.  0 (default): all blocks in one batch.  Results are identical (the blocks do not
 * interact, R13).  The environment variable MSPCG_GROUP sets the default of new contexts.  Errors: MSPCG_EINVAL (G < 0). */
int mspcg_set_block_group(mspcg_ctx* ctx, int blocks_per_group);

/* Fixed-point storage of PAPER.md:268-285 eq. 17 (reading R21: integer-limit 2^(bits-1) - 1, scale = largest |real| of the
 * colour-spinor's 24 numbers in fp32, integer = round-half-even(x / scale * limit) in fp32).
 * mspcg_fixed_pack / _unpack: the format itself.  abi_dev (DEVICE, fp64, ABI layout, Ls*V4/2*24 doubles) <-> q_dev (DEVICE, Ls*V4/2*24 signed
 * integers of `bits` = 8 or 16 bits, same order) and scale_dev (DEVICE, Ls*V4/2 floats, one per colour-spinor (s, x_cb)); unpack returns
 * integer / limit * scale evaluated in fp32.  Need no workspace and no gauge field.  Integers and scales are bit-identical to the oracle's.
 * mspcg_set_fixed_storage(bits = 8 | 16): the full-Ls preconditioner with fp32 inner storage (inner_prec = MSPCG_F32) passes every vector its
 * inner CG writes -- r, p, q = A p, x ("the matrix multiplication and BLAS operations use the 8-bit and 16-bit fixed-point
 * formats") -- through that store, inside the kernels that write them; <p, q> and |r|^2 are taken from the stored values.  The VALUES are those
 * of fixed-point storage; the bytes in HBM stay fp32 (a numerics mode for the paper's 8- vs 16-bit comparison, not a bandwidth one: DESIGN.md
 * section 9 says why the tensor-core hop cannot use the format).  bits = 0 (default): off.  Ignored by fp16 / fp64 inner storage and by the
 * reduced-Ls preconditioner.  Errors: MSPCG_EINVAL (null pointer, bits not in the list). */
int mspcg_fixed_pack(mspcg_ctx* ctx, const double* abi_dev, void* q_dev, float* scale_dev, int bits, void* stream);
int mspcg_fixed_unpack(mspcg_ctx* ctx, const void* q_dev, const float* scale_dev, double* abi_dev, int bits, void* stream);
int mspcg_set_fixed_storage(mspcg_ctx* ctx, int bits);

/* Host-only self check of the site tiles of the fp16 tile kernel (hop_tile.cuh; needs no GPU and no workspace): builds the tile tables of
 * the Dirichlet-block and the full-lattice geometry and verifies them against the neighbour tables (every output site in exactly one
 * tile, every neighbour's shared-memory slot holding that neighbour's column, absent neighbours on the zero column, copy runs consecutive
 * and complete).  out_host[8] (HOST): [0] 0 or a failure code, [1..4] tiles per block of kernel 2, kernel 4, kernels 3/5 (interior), kernel 3
 * (halo), [5..7] staged input columns per output site (8 without reuse) for kernel 4, for kernels 3/5, for the full lattice.
 * Errors: MSPCG_EINVAL (null pointer, or inconsistent tables: see mspcg_last_error). */
int mspcg_tile_check(mspcg_ctx* ctx, double out_host[8]);

/* Counters for reports: kernels launched by this context since creation. */
long mspcg_launch_count(const mspcg_ctx* ctx);

/* Per-kernel device timing for roofline reports.  mspcg_timing(ctx, 1) makes every later launch of the operator
 * kernels record a CUDA-event pair on its stream; mspcg_timing_read synchronises the device, sums the elapsed
 * milliseconds and launch counts per class into ms_host[10], launches_host[10] (HOST) and clears the record.
 * class = 5*geometry + kind;  geometry 0 = whole lattice, 1 = Dirichlet blocks;  kind 0 = Mphi (kernel 1 of eq. 16),
 * 1 = fused hop with one 5D matrix (kernels 2 and 4), 2 = fused hop of kernel 3, 3 = fused hop of kernel 5 (+dot),
 * 4 = BLAS-1 of the inner CG.  Off by default; timed benchmark regions run with it off. */
int mspcg_timing(mspcg_ctx* ctx, int enable);
int mspcg_timing_read(mspcg_ctx* ctx, double* ms_host, long* launches_host);

/* The two inner products of the Polak-Ribiere beta (eq. 18, R16) WITHOUT a context, a workspace or any allocation:
 * for callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops).  out_dev[0] = sum_i a[i] b[i],
 * out_dev[1] = sum_i a[i] c[i] (0 if c_dev is NULL) over n_reals doubles; a_dev, b_dev, c_dev (DEVICE, fp64, any layout: the sum runs over all
 * reals; a == b gives |a|^2), out_dev (DEVICE, 2 doubles, caller-owned).  Stream-ordered on `stream`, no synchronisation, no
 * cudaMalloc / cudaFree / allocating library call; one cudaMemsetAsync (4 bytes) and one kernel.  The partial sums (one pair per 16384
 * reals) and a ticket counter live in a file-scope device array of 513 KiB that every GPU holds from the time the library is loaded until
 * exit; hence n_reals <= mspcg_dot2_noalloc_max_reals() = 2^29 (a 4 GiB vector; C1..C4 fit, C5 does not).  The sums are added in a fixed
 * order: the result does not depend on the grid or on scheduling (bitwise equal from call to call).  ALL calls on a device share the
 * array: calls that overlap on the GPU (different streams without an ordering between them, or several host threads) RACE; calls on
 * one stream, or otherwise ordered, do not.  Errors: MSPCG_EINVAL (null out; null a or b with n_reals > 0; n_reals < 0 or above the maximum), MSPCG_ECUDA;
 * the message is mspcg_noalloc_last_error() (per host thread). */
int mspcg_dot2_noalloc(const double* a_dev, const double* b_dev, const double* c_dev, long n_reals, double* out_dev, void* stream);
long mspcg_dot2_noalloc_max_reals(void);
const char* mspcg_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MSPCG_H */
