/*
 * rpy_rigid.h -- C ABI of the rigid-multiblob layer around the mobility matvec (SURVEY.md 8(f)
 * rows N1, N2, N4): the kinematic matrix K and its transpose, the block-diagonal preconditioner, the
 * preconditioned GMRES solve of the mobility problem (one or several right-hand sides), and blob
 * positions from body poses.  Same library as rpy_matvec.h
 * (librpy_matvec.so), same conventions: plain device / host pointers, no allocation, no state,
 * errors as return codes, sm_100a only, no CPU fallback.
 *
 * The operations (arXiv:1602.02170; line numbers are /root/reference/PAPER.md):
 *
 *   K U         blob velocities of rigid motion, (K U)_i = u_p + omega_p x (r_i - q_p) for the blobs
 *               i of body p                                               Eqs. (2)-(3)
 *   K^T lambda  total force and torque per body, f_p = sum_i lambda_i,
 *               tau_p = sum_i (r_i - q_p) x lambda_i                       Eq. (10)
 *   P^-1        the indefinite block-diagonal preconditioner of Eq. (18): solve Eq. (19),
 *               [M~ -K; -K^T 0][lambda; U] = [x; y], with M~ the diagonal blocks M^(pp) of Eq. (17)
 *               (each body alone, with or without the wall), through the dense inverse of every
 *               M^(pp), formed from its Cholesky factor ("dense matrix inversion (e.g., Cholesky
 *               factorization)"), and the 6x6 body mobilities
 *               N~_pp = (K_p^T (M^(pp))^-1 K_p)^+                          PAPER.md:228-250
 *               (pseudo-inverse: a straight line of blobs or a single blob cannot resist
 *               a torque about its axis; that direction gets zero mobility, and the loads handed to
 *               the solve must then carry no torque about it)
 *   solve       Eq. (11), [M -K; -K^T 0][lambda; U] = [slip; -F], by right-preconditioned
 *               restarted GMRES
 *
 * Bodies are contiguous runs of blobs: body p owns blobs offsets[p] .. offsets[p+1]-1
 * (offsets[0] = 0, offsets[n_bodies] = n_blobs, every body has >= 1 blob and at most
 * RPY_RIGID_MAX_BODY_BLOBS) and has the tracking point q[p].  Rigid motions and force/torque pairs
 * are stored [n_bodies][6] = (u_p, omega_p) / (f_p, tau_p).  A solver vector is the concatenation
 * [lambda (3 n_blobs doubles, blob-major) ; U (6 n_bodies doubles)].
 *
 * Everything in this header is double precision, except that the solve can run its O(N^2) matvec
 * through the fp32 path of rpy_matvec.h (matvec_prec = RPY_PREC_F32_ACC64: the iterate is rounded
 * to float for the product and the residual stalls near 1e-6; "single precision can be used for
 * lower accuracy requirements").
 */
#ifndef RPY_RIGID_H
#define RPY_RIGID_H

#include "rpy_matvec.h"

#ifdef __cplusplus
extern "C" {
#endif

#define RPY_RIGID_MAX_BODY_BLOBS 1024
#define RPY_RIGID_MAX_RESTART 128
#define RPY_RIGID_MAX_BATCH 8

/* Additional status (values continue rpy_status): the Cholesky factorisation of some M^(pp) met a
 * non-positive pivot (a blob overlapping the wall, or coincident blobs). */
#define RPY_ERR_NOT_SPD 6

/* Third value of matvec_prec accepted by the solve only: fp32 products inside every GMRES cycle, an
 * fp64 product for the residual a later cycle starts from.  "Krylov methods ... allow one to lower the
 * accuracy of the matrix-vector product as the residual is reduced": a cycle that starts
 * from the TRUE residual rho ends with a true residual within margin = 1e-4 * rho of its Arnoldi estimate
 * (the fp32 product's error on the cycle's correction: a few eps_fp32 x cond(M); measured 0.3e-5 .. 2.2e-5).
 * While margin > tol / 2 a cycle ends when its estimate has dropped by 1e-4 (or to tol / 2e-4, from where the
 * next cycle can finish), x is updated and the fp64 residual of Eq. (11) is recomputed; once margin <= tol / 2
 * the cycle runs until estimate <= tol - margin and the solve returns without another fp64 product
 * (tol = 1e-8: two cycles, ONE fp64 product).  *h_rel_resid is then estimate + margin, an upper bound of
 * the true relative residual; when the solve stops after an fp64 residual (max_iter) it is that residual. */
#define RPY_PREC_MIXED 2

/* out[i] = beta * out[i] + alpha * (K U)_i.   beta == 0 overwrites (out may be uninitialised).
 *   d_pos [n_blobs][3], d_q [n_bodies][3], d_offsets [n_bodies+1] (int64), d_U [n_bodies][6],
 *   d_out [n_blobs][3] : device.  One warp per body.                                              */
rpy_status rpy_rigid_K_apply(int64_t n_blobs, int64_t n_bodies, const double *d_pos, const double *d_q,
                             const int64_t *d_offsets, const double *d_U, double alpha, double beta,
                             double *d_out, void *cuda_stream);

/* out[p] = beta * out[p] + alpha * (K^T lambda)_p;  d_lambda [n_blobs][3], d_out [n_bodies][6].
 * One warp per body, fixed summation order (bit-reproducible).                                    */
rpy_status rpy_rigid_KT_apply(int64_t n_blobs, int64_t n_bodies, const double *d_pos, const double *d_q,
                              const int64_t *d_offsets, const double *d_lambda, double alpha, double beta,
                              double *d_out, void *cuda_stream);

/* Bytes of device memory the preconditioner of these bodies needs (host arithmetic on the HOST
 * array h_offsets [n_bodies+1]); 0 if the offsets are not a valid partition.  Per body with
 * m = 3 * blobs: m*m doubles (the full symmetric inverse of M^(pp)), m*6 (Y = (M^(pp))^-1 K_p),
 * 36 (N~_pp), plus tables.  */
size_t rpy_rigid_precond_bytes(int64_t n_bodies, const int64_t *h_offsets);

/* Builds the preconditioner: for every body the dense M^(pp) (wall != 0: wall-corrected tensor,
 * else free space -- the "unbounded" preconditioner of Table III), its explicit inverse
 * ("dense matrix inversion"), Y = (M^(pp))^-1 K_p and N~_pp = (K_p^T Y)^+ (a
 * pseudo-inverse, taken with lengths in units of `a` so that it does not depend on the unit of length).
 * One CTA per body.  Bodies of up to 42 blobs (3*blobs <= 128): a register-resident block sweep of the
 * augmented matrix [M K; K^T 0] that yields all three in one pass; larger bodies: Cholesky factorisation,
 * L^-1 and L^-T L^-1 in place, in shared memory when 3*blobs <= 162, else in the body's slot of d_precond.
 * h_offsets is read before the call returns.
 * d_precond: device, 256-byte aligned, >= rpy_rigid_precond_bytes().  Synchronises the stream once (after
 * copying the offset tables up, before the build kernels are enqueued); a body that is not positive definite
 * is recorded in d_precond (its header names the first one) and reported by rpy_rigid_precond_info / the solve. */
rpy_status rpy_rigid_precond_build(int wall, int64_t n_blobs, int64_t n_bodies, const double *d_pos,
                                   const double *d_q, const int64_t *h_offsets, double a, double eta,
                                   void *d_precond, size_t precond_bytes, void *cuda_stream);

/* Copies the header of d_precond down (40 bytes; d_precond is only read), synchronises the stream and writes to
 * *h_first_bad_body the smallest body index whose factorisation (or 6x6 inversion) failed, or -1.  Returns
 * RPY_ERR_NOT_SPD in the former case, RPY_ERR_ARG when d_precond was not built for n_bodies bodies.          */
rpy_status rpy_rigid_precond_info(int64_t n_bodies, const void *d_precond, int64_t *h_first_bad_body,
                                  void *cuda_stream);

/* [lambda; U] = P^-1 [x; y]: Eq. (19) for every body.  d_in, d_out: solver vectors
 * (3 n_blobs + 6 n_bodies doubles), d_out must not overlap d_in.  One warp per body (four below 2,048 bodies):
 * t = (M^(pp))^-1 x (dense symmetric product), U = -N~ (y + Y^T x), lambda = t + Y U.
 * No host round trip, so a d_precond that was not built for (n_bodies, n_blobs) cannot be returned as a status:
 * the kernel then fills d_out with NaN (the solve checks the header on the host and returns RPY_ERR_ARG).  */
rpy_status rpy_rigid_precond_apply(int64_t n_blobs, int64_t n_bodies, const void *d_precond,
                                   const double *d_in, double *d_out, void *cuda_stream);

/* Copies out pieces of a built preconditioner (tests, diagnostics): for body p, the inverse
 * (M^(pp))^-1 (row-major m x m, symmetric) to d_inverse if non-NULL, and the 6x6 N~_pp (row-major)
 * to d_body_mobility if non-NULL.  Device to device, stream ordered.                               */
rpy_status rpy_rigid_precond_get(int64_t n_bodies, const int64_t *h_offsets, const void *d_precond,
                                 int64_t body, double *d_inverse, double *d_body_mobility,
                                 void *cuda_stream);

/* Blob positions of identical bodies from their poses (footnote 4: "only the positions
 * and orientations of the rigid bodies (so only up to 7 numbers per body) need to be communicated to
 * the GPU"):  r_{p,t} = c_p + R(theta_p) template_t,  blob index p * blobs_per_body + t.
 *   d_template [blobs_per_body][3] reference configuration, d_centres [n_bodies][3],
 *   d_quats [n_bodies][4] unit quaternions (s, p1, p2, p3) (normalised again inside),
 *   d_pos [n_bodies * blobs_per_body][3] overwritten.  Element type per `prec` (double / float).   */
rpy_status rpy_rigid_blob_positions(rpy_prec prec, int64_t n_bodies, int blobs_per_body, const void *d_template,
                                    const void *d_centres, const void *d_quats, void *d_pos, void *cuda_stream);

/* Workspace of the solve: restart+1 Krylov vectors, four work vectors, the matvec workspace (of the fp64
 * product too when matvec_prec is not RPY_PREC_F64: such solves form fp64 residuals) and, for fp32 products,
 * float copies of positions, iterate and product.                                                  */
size_t rpy_rigid_solve_workspace_bytes(rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies, int restart);

/* Optional extras of the solve (pass NULL for none).  The library creates no CUDA object of its own:
 *   side_stream, side_event   a second cudaStream_t and a cudaEvent_t (timing may be disabled) of the
 *       caller.  With them the host reads the outcome of iteration j on side_stream, ordered after that
 *       iteration by side_event, while `cuda_stream` already runs iteration j+1; without them it reads on
 *       `cuda_stream` and the device idles while the next iteration is being enqueued.
 *   shard, n_shards, reduce, reduce_ctx   multi-GPU (one process per GPU, all arguments replicated): rank
 *       `shard` of `n_shards` computes its share of every product M lambda (rpy_*_matvec_shard's unordered
 *       tile pairs) and calls reduce(reduce_ctx, d_buf, count, cuda_stream) once per product; the hook must
 *       make d_buf[0..count) (doubles, device) the SUM over all ranks, in stream order on cuda_stream (e.g.
 *       an in-place NCCL all-reduce), and return 0.  Everything else of the iteration is replicated, so the
 *       ranks take the same decisions.  n_shards > 1 needs n_rhs == 1 and n_blobs >= 1,152.              */
typedef int (*rpy_reduce_fn)(void *reduce_ctx, double *d_buf, int64_t count, void *cuda_stream);
typedef struct rpy_rigid_solve_ext {
    void *side_stream;
    void *side_event;
    int shard;
    int n_shards;               /* 0 or 1: the whole product on this GPU */
    rpy_reduce_fn reduce;
    void *reduce_ctx;
} rpy_rigid_solve_ext;

/* Solves the mobility problem, Eq. (11), for lambda and U given the applied forces/torques F and an
 * optional slip velocity, by right-preconditioned GMRES(restart) from a zero initial guess: the
 * iteration stops when the residual of (11) is <= tol * ||[slip; -F]|| (Table III: tol = 1e-8,
 * PAPER.md:680) or after max_iter matrix applications.  One iteration = P^-1 (above), the O(N^2)
 * product M lambda (rpy_wall_matvec / rpy_free_matvec with matvec_prec), K, K^T, classical
 * Gram-Schmidt applied twice, a Givens update of the small Hessenberg problem and the stopping test --
 * all on the device (seven launches).  The host reads 80 bytes per iteration to follow the device's
 * decision and to fill h_history, so the call SYNCHRONISES; see rpy_rigid_solve_ext for how that read
 * is kept off the critical path.
 *   wall        != 0: wall-corrected M in the product (the preconditioner is whatever was built)
 *   matvec_prec RPY_PREC_F64; RPY_PREC_F32_ACC64 (fp32 products; converges on the fp32 operator's residual
 *               estimate, then ONE fp64 product gives the true residual that is reported); RPY_PREC_MIXED
 *   d_F         [n_bodies][6] device;  d_slip [n_blobs][3] device or NULL (zero slip)
 *   d_lambda    [n_blobs][3], d_U [n_bodies][6] : device, overwritten
 *   h_history   host, max_iter+1 doubles or NULL: relative residual after each iteration, [0] = 1
 *   h_n_iter    host, matrix applications used;  h_rel_resid host, final relative residual: with
 *               RPY_PREC_F64 the Arnoldi estimate, which IS the residual of the operator used; with
 *               RPY_PREC_F32_ACC64 the true residual of Eq. (11) (one fp64 product at the end); with
 *               RPY_PREC_MIXED an upper bound of the true residual (see RPY_PREC_MIXED; a caller who wants the
 *               residual itself applies rpy_rigid_saddle_apply to the solution)
 * Returns RPY_OK also when max_iter was reached without convergence (check *h_rel_resid).
 * A d_precond that was not built for these bodies (n_bodies, n_blobs) is RPY_ERR_ARG.                */
rpy_status rpy_rigid_mobility_solve(int wall, rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies,
                                    const double *d_pos, const double *d_q, const int64_t *d_offsets,
                                    const double *d_F, const double *d_slip, double a, double eta,
                                    const void *d_precond, double tol, int restart, int max_iter,
                                    double *d_lambda, double *d_U,
                                    double *h_history, int *h_n_iter, double *h_rel_resid,
                                    void *d_workspace, size_t workspace_bytes, void *cuda_stream,
                                    const rpy_rigid_solve_ext *ext);

/* The same for n_rhs (1..RPY_RIGID_MAX_BATCH) right-hand sides at once -- e.g. the columns of the body
 * mobility matrix N of Eq. (12), one unit force or torque each.  n_rhs independent GMRES processes
 * advance in lockstep and share every launch, in particular ONE product call with n_rhs right-hand
 * sides per iteration (the multi-right-hand-side kernel builds each pair tensor once for all of them:
 * 46 + 10 n_rhs FP-pipe operations per pair instead of 33 per pair and right-hand side).  The iteration
 * stops when EVERY right-hand side has reached tol (or at max_iter); a zero right-hand side gives zero.
 *   d_F [n_rhs][n_bodies][6], d_slip [n_rhs][n_blobs][3] or NULL, d_lambda [n_rhs][n_blobs][3],
 *   d_U [n_rhs][n_bodies][6];  h_history NULL or [n_rhs][max_iter+1];  h_rel_resid [n_rhs];
 *   workspace: rpy_rigid_solve_batch_workspace_bytes().                                            */
size_t rpy_rigid_solve_batch_workspace_bytes(rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies, int restart,
                                             int n_rhs);
rpy_status rpy_rigid_mobility_solve_batch(int wall, rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies, int n_rhs,
                                          const double *d_pos, const double *d_q, const int64_t *d_offsets,
                                          const double *d_F, const double *d_slip, double a, double eta,
                                          const void *d_precond, double tol, int restart, int max_iter,
                                          double *d_lambda, double *d_U,
                                          double *h_history, int *h_n_iter, double *h_rel_resid,
                                          void *d_workspace, size_t workspace_bytes, void *cuda_stream,
                                          const rpy_rigid_solve_ext *ext);

/* The operator of Eq. (11) alone: out = [M lambda - K U ; -K^T lambda] for a solver vector
 * in = [lambda; U] (tests; residual checks).  d_workspace as for the solve with restart = 1.      */
rpy_status rpy_rigid_saddle_apply(int wall, rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies,
                                  const double *d_pos, const double *d_q, const int64_t *d_offsets,
                                  double a, double eta, const double *d_in, double *d_out,
                                  void *d_workspace, size_t workspace_bytes, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* RPY_RIGID_H */
