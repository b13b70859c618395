/* rpy_bench_aids.h -- measurement aids of bench.py.  NOT part of the product: the method's C ABI is
 * include/rpy_matvec.h and include/rpy_rigid.h; nothing here computes a mobility.  Built as
 * bench_aids/librpy_bench_aids.so (python -m bench_aids), which links against the product library
 * only for rpy_bench_matvec_phases.                                                              */
#ifndef RPY_BENCH_AIDS_H
#define RPY_BENCH_AIDS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* Register-only chains of independent fused multiply-adds (or MUFU.RSQ) on every SM, timed with CUDA
 * events on `cuda_stream` (which is synchronised): the denominator of the ALU roofline (DESIGN.md
 * "Roofline") measured on the GPU and at the clocks the bench runs at.  *h_elapsed_ms: duration;
 * *h_fma_count: scalar (lane) operations executed.
 *   kind 0 FFMA, 1 packed FFMA2, 2 DFMA (loop-invariant multiplier and addend registers),
 *        3 MUFU.RSQ, 4 FFMA2 / 5 FFMA with three distinct register operands per instruction.
 * d_sink: >= 8 bytes of device memory (defeats dead-code elimination).
 * Returns 0, or 1 (NULL pointer), 2 (bad kind / iters), 5 (CUDA error).                          */
int rpy_bench_pipe_probe(int kind, int iters, void *d_sink, float *h_elapsed_ms, double *h_fma_count,
                         void *cuda_stream);

/* What an FP-pipe instruction costs by the form of its operands (the all-pairs kernels are bound
 * by the delivery of register operands, not by the pipe itself).  12 independent accumulators per thread, 128 threads per
 * CTA, `ctas_per_sm` (1..4) CTAs per SM; operands are loaded once from d_scratch (zeros) as 64-bit words.
 *   kind 0 FFMA2 acc = x*x + acc          two distinct register pairs
 *        1 FFMA2 acc = x*1.5 + acc        two pairs and an immediate
 *        2 FFMA2 acc = x*y' + acc         three distinct pairs, none shared with the neighbouring instructions
 *        3 FFMA2 acc = x*y0 + acc         three distinct pairs, one the same for all (served by the operand-reuse cache)
 *        4 FFMA2 acc = x*s + acc          two pairs and a 32-bit scalar operand (.F32 broadcast form)
 *        5, 6, 7 DFMA                     as 0, 2, 3
 * d_scratch: >= 8 + 8 * 128 * 4 * 12 bytes of zeroed device memory.  *h_lane_ops: scalar (lane) operations executed.
 * Returns 0, or 1 (NULL pointer), 2 (bad argument), 5 (CUDA error).                                               */
int rpy_bench_operand_probe(int kind, int ctas_per_sm, int iters, void *d_scratch, float *h_elapsed_ms,
                            double *h_lane_ops, void *cuda_stream);

/* FP64 pipe beside the FP32 pipe: 8 CTAs of 128 threads per SM, of which `n64_per_sm` (0..8) run DFMA
 * chains of `iters64` steps and the others FFMA2 chains of `iters32` steps (role by arrival order on
 * the SM).  three_reg != 0: three distinct register operands per instruction.  Outputs: duration and
 * the lane operations of each kind.  d_scratch: >= 1032 bytes of device memory.                  */
int rpy_bench_coissue_probe(int n64_per_sm, int iters32, int iters64, int three_reg, void *d_scratch,
                            float *h_elapsed_ms, double *h_ops32, double *h_ops64, void *cuda_stream);

/* rpy_wall_matvec / rpy_free_matvec (wall != 0 / == 0; same arguments, checks and result; n_blobs >= 1)
 * with four caller-owned CUDA events (cudaEvent_t as void*) recorded on `cuda_stream`:
 *   [0] before prepack, [1] before the all-pairs kernel, [2] after it, [3] after finalise
 * of the first right-hand-side group (n_rhs <= 8: the only one).  prec: 0 fp64, 1 fp32 path.
 * Returns the product's rpy_status.                                                              */
int rpy_bench_matvec_phases(int wall, int prec, int64_t n_blobs, int n_rhs, const void *d_pos,
                            const void *d_force, void *d_vel, double a, double eta, void *d_workspace,
                            size_t workspace_bytes, void *cuda_stream, void *const *cuda_events4);

#ifdef __cplusplus
}
#endif
#endif
