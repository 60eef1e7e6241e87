/*
 * tsm.h -- C ABI of the B200-native truncated-solver-method (TSM) loop library.
 *
 * The calls follow the paper's statement of the problem (arXiv:1211.0126; line numbers
 * are /root/reference/PAPER.md, "Ax/Ox/Cx" are the readings listed in DESIGN.md):
 *   - noise sources |eta_j> with Z2/Z4 components          (Eq. 2.1)
 *   - solve M|s_j> = |eta_j>                               (Eq. 2.2)
 *   - high precision, or truncated "at a large residual or equivalently a fixed
 *     number of iterations"
 *   - loops (1/N) sum <eta^dag X s> for all insertion times
 *   - the TSM combination                                  (Eq. 2.4)
 *
 * Conventions
 *   - Every call returns an int status: TSM_OK or a negative TSM_E* code.  Nothing throws
 *     or aborts.  tsm_last_error() gives a human-readable message for the last failure.
 *   - Pointers named host_* are HOST memory, dev_* are DEVICE memory on the context's GPU.
 *     Host arrays are caller-owned fp64 in lexicographic layouts (C1, C2):
 *       lex(x) = x0 + L0*(x1 + L1*(x2 + L2*x3)), x = (x,y,z,t);
 *       spinor  [lex][alpha 0..3][colour 0..2][re,im];
 *       links   [mu 0..3][lex][row c][col c'][re,im], (U psi)_c = sum_c' U_cc' psi_c';
 *       loops   [op][t][re,im], op = 0..15 the 16 Gamma of C3 (1, g5, g_mu, g5 g_mu,
 *               sigma_01,02,03,12,13,23), then (TSM_OPS_DERIVATIVE) 16 + 16*mu + Gamma for the derivative
 *               loops, then (TSM_OPS_ONE_END) 16 more: the one-end loops of Eq. 2.5,
 *               L1_Gamma(t) = -2 i (2 kappa mu) sum_{x in t} s^dag gamma5 Gamma s, whose noise average is
 *               sum_{x in t} tr[Gamma (M_u^-1 - M_d^-1)(x,x)] (kappa-normalised operators), then
 *               (TSM_OPS_GEN_ONE_END) 16 more: Eq. 2.6, L2_Gamma(t) = 2 sum_{x in t} s^dag gamma5 Gamma gamma5 D_W s,
 *               D_W = 1 - kappa D_hop, noise average sum_{x in t} tr[Gamma (M_u^-1 + M_d^-1)(x,x)].
 *   - The library allocates no large device memory.  All of it (link copies, solver
 *     vectors, solution slots, reduction scratch) lives in ONE caller-provided workspace
 *     (a torch tensor's data_ptr()), sized by tsm_workspace_bytes().  The context owns
 *     only metadata, a few KB of pinned host memory and a few KB of device scalars.
 *   - Work is enqueued on the stream given to tsm_set_stream().  By default, and when that call is given
 *     NULL, the library uses a BLOCKING stream of its own: it is ordered with the caller's legacy default
 *     stream exactly as default-stream work would be, and unlike the legacy stream it can be captured, which
 *     lets the solver run its CG iterations as a cached CUDA graph (tsm_set_graphs).  Calls that return host scalars or arrays synchronise that stream
 *     before returning; calls that only take dev_* pointers are asynchronous.
 *   - "Native layout" of a single-parity spinor field with V_h = V/2 sites, nrhs sources:
 *       [rhs][block of 32 cb sites][chunk][site in block] of 16-byte vectors (V_h is padded up
 *       to a multiple of 32; the padding is never read or written); fp64: 12 chunks of double2
 *       (one complex each, q = 3*alpha + c); fp32: 6 chunks of float4 (complex q = 2*chunk,
 *       2*chunk+1); bf16: 3 chunks of 8 x bf16 (complex q = 4*chunk .. 4*chunk+3);
 *       cb = lex >> 1 is the checkerboard index, parity = (x+y+z+t) & 1 (H1).
 *       A full-lattice field is [parity 0,1] of those.  tsm_field_bytes() gives sizes.
 *   - Error behaviour: wrong-state calls (no workspace / gauge / params yet) -> TSM_ESTATE;
 *     bad dims, enum, nrhs, slot or NULL pointer -> TSM_EINVAL; CUDA failure -> TSM_ECUDA.
 */
#ifndef TSM_H
#define TSM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tsm_ctx tsm_ctx; /* opaque; owned by the library */

enum { TSM_OK = 0, TSM_EINVAL = -1, TSM_ESTATE = -2, TSM_ECUDA = -3, TSM_ENOTUNITARY = -4,
       TSM_EBREAKDOWN = -5, TSM_ENOCONV = -6 };
enum { TSM_F64 = 0, TSM_F32 = 1, TSM_BF16 = 2,           /* spinor storage precision */
       TSM_MIXED = 3 };  /* tsm_solve only: fp64 defect correction around the fp32 CG (fp64 solution, tol > 0) */
enum { TSM_Z4 = 0, TSM_Z2 = 1 };                           /* noise kind (A5)          */
enum { TSM_OP_D_EO = 0,      /* out_e = D_eo in_o                         (H5)           */
       TSM_OP_D_OE = 1,      /* out_o = D_oe in_e                                        */
       TSM_OP_MHAT = 2,      /* out_e = (R - kappa^2 D_eo R^-1 D_oe) in_e (O4)           */
       TSM_OP_MHAT_DAG = 3,  /* out_e = Mhat^dagger in_e                                 */
       TSM_OP_M_FULL = 4 };  /* out = M in on the full lattice, [parity] fields (O2)     */
#define TSM_MAX_NRHS 16
#define TSM_N_LOCAL_OPS 16
#define TSM_N_DERIV_OPS 64
#define TSM_N_ONE_END_OPS 16
#define TSM_N_GEN_ONE_END_OPS 16
#define TSM_MAX_MOMENTA 16
#define TSM_MAX_OPS (TSM_N_LOCAL_OPS + TSM_N_DERIV_OPS + TSM_N_ONE_END_OPS + TSM_N_GEN_ONE_END_OPS + 16 * TSM_MAX_MOMENTA)
/* which loops are computed besides the 16 local ones (bit mask `ops` of tsm_loops_reset / tsm_run_loop_set) */
enum { TSM_OPS_DERIVATIVE = 1,   /* one-derivative loops, 4 directions (O6b)                 */
       TSM_OPS_ONE_END = 2,      /* one-end-trick loops of Eq. 2.5; need tsm_set_params   */
       TSM_OPS_GEN_ONE_END = 4,  /* generalised one-end-trick loops of Eq. 2.6; same      */
       TSM_OPS_MOMENTA = 8 };    /* momentum-projected local loops for the list of tsm_loops_set_momenta   */

/* Geometry (H1).  dims = (Lx,Ly,Lz,Lt), every extent even and >= 4.  t_boundary = +1
 * periodic or -1 antiperiodic in time (A3).  device = CUDA ordinal. */
int tsm_create(tsm_ctx** out, const int dims[4], int t_boundary, int device);
int tsm_destroy(tsm_ctx* ctx);
const char* tsm_last_error(const tsm_ctx* ctx);

/* Bytes of one single-parity native field of `nrhs` sources in precision `prec`. */
size_t tsm_field_bytes(const tsm_ctx* ctx, int prec, int nrhs);

/* Workspace: bytes needed for up to max_nrhs simultaneous sources in a context whose widest spinor precision is
 * `prec`: TSM_F64 = everything (fp64 and fp32 link copies, fp64-sized solver vectors and solution
 * slots, staging for host<->device conversion); TSM_F32 = a low-precision-only workspace for fp32 / bf16-storage
 * solves (no fp64 link copy, vectors and slots sized for fp32: about half the bytes) -- on it fp64 / mixed solves,
 * fp64 stencils and the fp64 true residual return TSM_ESTATE.  Any other `prec` is an error (0 bytes / TSM_EINVAL).
 * The pointer must be 256-byte aligned device memory that outlives every later call. */
size_t tsm_workspace_bytes(const tsm_ctx* ctx, int max_nrhs, int prec);
int tsm_set_workspace(tsm_ctx* ctx, void* dev_ptr, size_t bytes, int max_nrhs, int prec);
int tsm_set_stream(tsm_ctx* ctx, void* cuda_stream);   /* a cudaStream_t; NULL = the library's own stream */

/* kappa, mu of the kappa-normalised twisted-mass operator of O2:
 * M = 1 + 2 i kappa mu gamma5 - kappa D_hop  (= 2 kappa x the paper's M_u). */
int tsm_set_params(tsm_ctx* ctx, double kappa, double mu);

/* H2: upload one gauge configuration.  host_links is [4][V][3][3][2] fp64,
 * copied (the caller keeps its array); it may be pinned or pageable.  The fp64 copy always
 * keeps 18 reals; `reconstruct` (18 or 12) selects the storage of the fp32 copy used by the
 * F32/BF16 paths (12: first two rows, third row rebuilt in-kernel, A22).  Links further than
 * 1e-10 from SU(3) give TSM_ENOTUNITARY when reconstruct == 12.  max_unitarity_dev (may be
 * NULL) receives max(|U^dag U - 1|_max, |det U - 1|). */
int tsm_set_gauge(tsm_ctx* ctx, const double* host_links, int reconstruct, double* max_unitarity_dev);

/* H3: generate noise source `source_id` of stream `seed` (O3: Philox4x32-10, counter
 * (lex, source_id, kind)) on the device and copy it to host_out [V][4][3][2] in lex order
 * (parity-test hook; the solver generates its sources itself). */
int tsm_noise(tsm_ctx* ctx, uint64_t seed, uint32_t source_id, int kind, double* host_out);

/* Host lex fp64 [nrhs][V][4][3][2]  <->  device native full-lattice field [parity][rhs][block][chunk][site]. */
int tsm_pack(tsm_ctx* ctx, int prec, int nrhs, const double* host_lex, void* dev_native);
int tsm_unpack(tsm_ctx* ctx, int prec, int nrhs, const void* dev_native, double* host_lex);

/* H5: one application of the stencil on caller buffers in native layout (asynchronous).
 * D_EO/D_OE/MHAT/MHAT_DAG take and give single-parity fields; M_FULL full-lattice fields.
 * dev_in and dev_out must not overlap. */
int tsm_dslash(tsm_ctx* ctx, int op, int prec, int nrhs, const void* dev_in, void* dev_out);

/* H3+H4+H6+H7: generate sources source_ids[0..nrhs) and solve M s = eta for all of them
 * at once by even-odd preconditioned CG on Mhat^dag Mhat (O4, O5; batched, not block, CG:
 * every source has its own alpha, beta, stopping iteration, A14).
 *   tol > 0 : stop source j at the first iteration with |r_k|/|b'| <= tol (A8); a source
 *             that has not got there after max_iter iterations reports TSM_ENOCONV.
 *   tol == 0: exactly max_iter iterations, no residual test (A9).
 * The full-lattice solutions stay in workspace slot `slot` (0 or 1), in precision `prec`
 * (BF16 solves leave fp32 solutions).  prec = TSM_MIXED (needs tol > 0) reaches the same fp64 solution as
 * TSM_F64 at low-precision cost: it stops on the TRUE fp64 residual |b' - A x|/|b'| <= tol of the
 * preconditioned normal system, corrections e come from fp32 CG solves of A e = r to 1e-5; `iters` is the
 * total of fp32 iterations, rel_resid_rec that true residual.  info (may be NULL) is a host array [nrhs];
 * rel_resid_true (the fp64 |eta - M s|/|eta| of the full system) is filled only when
 * want_true_resid != 0.  Returns TSM_OK if every source ended TSM_OK, else the first
 * non-OK per-source status (solutions are kept either way). */
typedef struct {
    int iters;              /* CG iterations done for this source              */
    int status;             /* TSM_OK, TSM_EBREAKDOWN (A13) or TSM_ENOCONV     */
    double rel_resid_rec;   /* sqrt(|r_k|^2/|b'|^2) of the CG recursion (A8)   */
    double rel_resid_true;  /* fp64 true residual of the full system, or -1    */
    double secs;            /* device time of the whole batch (same for all j) */
} tsm_solve_info;
int tsm_solve(tsm_ctx* ctx, uint64_t seed, const uint32_t* source_ids, int nrhs, int kind,
              int prec, double tol, int max_iter, int slot, int want_true_resid,
              tsm_solve_info* info);
/* tsm_solve without the wait: tsm_solve_async only ENQUEUES the solve on the context's stream (no host synchronisation:
 * in residual mode the stopping test runs on the device, tsm_set_graphs mode 2; TSM_MIXED still reads its outer-loop
 * state on the host) and returns TSM_OK or an argument / state error; the slot may be used by later calls on the same
 * stream (tsm_loops_add_lp, ...) at once.  tsm_solve_wait synchronises and reports on the solve LAST enqueued into
 * `slot` exactly as tsm_solve would have (TSM_ESTATE if none is pending).  tsm_solve == tsm_solve_async with host
 * polling allowed + tsm_solve_wait; the iterates are bit-identical. */
int tsm_solve_async(tsm_ctx* ctx, uint64_t seed, const uint32_t* source_ids, int nrhs, int kind, int prec, double tol,
                    int max_iter, int slot);
int tsm_solve_wait(tsm_ctx* ctx, int slot, int want_true_resid, tsm_solve_info* info);

int tsm_get_solution(tsm_ctx* ctx, int slot, int rhs, double* host_out /* [V][4][3][2] */);
/* Overwrite the solution held in a slot (contraction parity with the oracle's s, A16(i));
 * the slot keeps the seed/source ids/kind/nrhs of the last tsm_solve into it. */
int tsm_set_solution(tsm_ctx* ctx, int slot, int rhs, const double* host_in /* [V][4][3][2] */);

/* H8-H10: per-timeslice loops and the TSM accumulators (Eq. 2.4, O6, O6b, O7).  `ops` is a bit mask of
 * TSM_OPS_*: n_ops = 16 [+ 64] [+ 16] [+ 16] [+ 16 nmom].  The one-end loops are bilinear in s, and Eq. 2.4 is applied to them
 * exactly as to the others: correction = L1(s_HP) - L1(s_LP), biased estimate = L1(s_LP). */
int tsm_loops_reset(tsm_ctx* ctx, int ops);
/* Momenta of the projected loops (Fourier transform of the loops; reading A25): n is [nmom][3]
 * integers, p_i = 2 pi n_i / L_i, nmom <= TSM_MAX_MOMENTA.  With TSM_OPS_MOMENTA in `ops` the op list ends with
 * 16 loops per momentum, op = base + 16*m + Gamma: sum_{x in t} exp(+i p.x) eta^dag Gamma s.  Call it before
 * tsm_loops_reset (which fixes n_ops). */
int tsm_loops_set_momenta(tsm_ctx* ctx, int nmom, const int* n);
int tsm_loops_add_correction(tsm_ctx* ctx, int slot_hp, int slot_lp); /* += L(HP)-L(LP); N_HP += nrhs */
int tsm_loops_add_lp(tsm_ctx* ctx, int slot_lp);                   /* += L(LP); N_LP += nrhs  */
int tsm_loops_source(tsm_ctx* ctx, int slot, int rhs, double* host_out /* [n_ops][Lt][2] */);
int tsm_loops_finalize(tsm_ctx* ctx, double* host_out /* [n_ops][Lt][2] */);
/* Accumulator access for checkpoint/resume (state = seed, next id, sums). */
int tsm_loops_get_state(tsm_ctx* ctx, double* host_corr, double* host_lp, int* n_hp, int* n_lp);
int tsm_loops_set_state(tsm_ctx* ctx, const double* host_corr, const double* host_lp, int n_hp, int n_lp);

/* Convenience driver: the whole of Eq. 2.4 for one gauge configuration.  Sources
 * 0..n_hp-1 get an HP (fp64, hp_tol) and an LP solve; sources n_hp..n_hp+n_lp-1 an LP solve
 * (lp_prec; lp_tol > 0 or exactly lp_iters iterations); batches of nrhs sources.
 * secs_out (may be NULL) receives the device time from the first noise kernel to the
 * final loops (reading A23). */
int tsm_run_loop_set(tsm_ctx* ctx, uint64_t seed, int kind, int n_hp, int n_lp, int lp_prec,
                     double lp_tol, int lp_iters, double hp_tol, int hp_max_iter, int nrhs,
                     int ops, double* host_out, double* secs_out);

/* Solver of the HP solves of tsm_run_loop_set ("high precision" inversions): TSM_MIXED (default:
 * fp64 defect correction around the fp32 CG, stopped on the fp64 TRUE residual -- the same fp64 solution at
 * low-precision bandwidth cost) or TSM_F64 (plain fp64 CG; what a workload that is "fp64 throughout" asks for). */
int tsm_set_hp_precision(tsm_ctx* ctx, int prec);

/* Name of the stencil kernel the library launches for spinor precision `prec` and a batch of `nrhs` sources in this
 * context (static string; measurement aid: bench.py prints it beside the roofline). */
const char* tsm_stencil_kernel_name(const tsm_ctx* ctx, int prec, int nrhs);

/* Tuning / test switches (no environment variables are read anywhere in the library).
 * tsm_set_stencil_kernel: 0 = automatic (default; on lattices of at most 16 384 sites per
 * parity every fp64 / fp32 stencil runs in k_dslash_small; otherwise fp64 and single sources use k_dslash and
 * fp32 / bf16 batches k_dslash_tile), 1 = k_dslash, 2 = k_dslash_tile (fp32 / bf16), 3 = k_dslash_box (fp32, lattice
 * permitting), 5 = k_dslash_small (fp64 / fp32).  A forced kernel that cannot serve a call falls back to the
 * automatic choice.  k_dslash and k_dslash_tile give a source bit-identical results; k_dslash_box and k_dslash_small
 * each differ from them in rounding, so a context should stay with one choice while results are being compared.  tsm_set_graphs: how the CG iterations are launched: 4 (default) = automatic: mode 3
 * on the lattices served by k_dslash_small (where it measures 34-42 % faster; there the same launch also does the
 * even-odd preparation, the CG start and the reconstruction of an fp64 / fp32 solve, so a solve is the noise kernel
 * plus ONE launch), mode 1 elsewhere; 1 = cached CUDA graphs
 * of 4 iterations, the host reads the all-done flag between them in residual mode; 2 = the whole iteration loop as
 * ONE graph launch, a WHILE node whose body is one captured iteration and whose condition (a source is still live
 * and the iteration budget is not used up) is set on the device by the last kernel of the body: no host round trip,
 * but measured 4.5 us per pass slower than mode 1 on this driver; 3 = the whole loop in ONE
 * cooperative launch of a persistent kernel (grid-wide barriers between the phases of an iteration, stopping test on
 * the device; fp64 / fp32, lattices of at most 131 072 sites per parity, other cases fall back to mode 1) whose
 * stencil arithmetic is that of the context's stencil kernel (k_dslash's with 128-site tiles, k_dslash_small's with
 * 32-site blocks); 0 = kernel by kernel.  All modes give bit-identical iterates for fp64 / fp32 sources (for a batch of
 * 2 or more fp32 sources with k_dslash_tile as the stencil, mode 3 agrees with it because k_dslash_tile and k_dslash do). */
int tsm_set_stencil_kernel(tsm_ctx* ctx, int which);
int tsm_set_graphs(tsm_ctx* ctx, int mode);

/* Measurement aid for the tensor-core clause of north_star (csrc/mma_probe.cu): times the only dense
 * contraction of the stencil -- per site and hop, G = U H with U one SU(3) link and H the 3 x 24 block of 12 sources'
 * projected half spinors -- on `nsites` (site, hop) pairs held in registers, repeated `inner` times per launch on
 * H + it * eps with G accumulated (so the arithmetic, not operand traffic, is timed), `reps` launches, in one formulation:
 * variant 0 packed fp32 FMAs (the stencil's own), 1 mma.sync TF32, 2 mma.sync 3xTF32, 3 fp64 FMAs, 4 fp64 mma.sync.
 * Outputs (host): microseconds per launch and the largest error relative to the largest fp64 reference value.
 * Allocates and frees its own small device buffers; blocks until done.  Not part of the hot path. */
int tsm_probe_su3_tensor(tsm_ctx* ctx, int variant, int nsites, int inner, int reps, double* us_per_launch, double* max_rel_err);

/* The one entry point that ALLOCATES NOTHING (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): the 16 local loops eta^dag Gamma s per timeslice (H8) of
 * `nrhs` sources whose solutions the caller holds on the device.  dev_solution: native full-lattice field
 * [parity][rhs][block of 32 sites][chunk][site] in precision `prec` (TSM_F64 or TSM_F32), as tsm_pack writes it;
 * source_ids: HOST array of nrhs ids (passed to the kernel by value); seed / kind: the noise of those sources (eta is
 * regenerated, never read); dev_loops: DEVICE output, [nrhs][16][Lt][2] doubles.  Needs no workspace, gauge field or
 * parameters; calls no cudaMalloc / cudaFree; enqueues two kernels on the context's stream and returns without
 * synchronising.  Its reduction scratch is a static device array of tsm_noalloc_scratch_bytes() = 4 MiB that every GPU
 * loading the library holds until exit: calls with nrhs * Lt * 2 * nblk * 32 doubles beyond that (nblk = number of
 * 1024-site pieces of a timeslice and parity, at most 8) return TSM_EINVAL.  All calls share the array: calls on one
 * stream are ordered, calls that overlap on the GPU (several streams or contexts on one device) race.  The result is
 * bit-identical to the local loops of tsm_loops_source. */
size_t tsm_noalloc_scratch_bytes(void);
int tsm_loops_local_noalloc(tsm_ctx* ctx, int prec, int nrhs, const void* dev_solution, uint64_t seed, const uint32_t* source_ids,
                            int kind, double* dev_loops);

/* Number of kernels this library has launched on the context since creation. */
long long tsm_launch_count(const tsm_ctx* ctx);

/* Measurement aid: with profiling enabled every stencil and CG
 * BLAS launch is bracketed by CUDA events on the library's stream.  tsm_profile_read
 * synchronises, returns the summed duration (ms) and the number of launches recorded so far
 * for one class and forgets them.  prec: TSM_F64/F32/BF16; kind: 0 stencil (H5), 1 stencil
 * with the x term, 2 stencil with x term and per-tile sum of |out|^2, 3 stencil with x term whose
 * result updates the CG residual in place (r -= alpha q, per-tile |r|^2), 4 the CG x/p update,
 * 5 / 6 / 7 / 8 / 9 the local / derivative / one-end / generalised one-end / momentum contraction (prec = that of the slot);
 * nrhs <= 0 matches any batch size. */
int tsm_profile(tsm_ctx* ctx, int enable);
int tsm_profile_read(tsm_ctx* ctx, int prec, int kind, int nrhs, double* total_ms, long long* count);

#ifdef __cplusplus
}
#endif
#endif /* TSM_H */
