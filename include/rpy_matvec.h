/*
 * rpy_matvec.h -- C ABI of the B200-native RPY / wall-RPY blob mobility matvec.
 *
 * The operation (arXiv:1602.02170; line numbers are /root/reference/PAPER.md):
 *
 *   u_i = sum_{j=0}^{N-1} M_ij lambda_j        all j, including j = i      Eq. (6)
 *
 * evaluated by direct O(N_b^2) summation on one GPU, where the
 * 3x3 block M_ij is
 *
 *   free space:  (1/(6 pi eta a)) RPY(r_i - r_j)                           Eq. (9)
 *   single wall: the same plus the translation-translation Rotne-Prager-Blake wall
 *                correction, i.e. Eq. (7) applied to the image part
 *                of the half-space Green's function; closed form and the
 *                readings taken where the paper is silent: DESIGN.md "Readings".
 *
 * The wall is the plane z = 0 (z is the third coordinate), the fluid is z > 0.  One
 * radius `a` and one viscosity `eta` for all blobs.  The tensor is only meaningful for
 * blob heights z >= a; heights are not checked by the matvec calls
 * (rpy_wall_count_below is the optional O(N) check).  r <= 2a takes the overlap branch
 * of Eq. (9); r = 0 (i = j or coincident blobs) gives M_ij = (6 pi eta a)^-1 I plus the
 * wall term.
 *
 * Conventions common to every entry point
 *  - "device" pointers are CUDA device pointers owned by the caller; "host" pointers
 *    are ordinary host memory (pinned memory makes the host calls faster, it is not
 *    required).  The library never allocates or frees memory and keeps no state between
 *    calls except the thread-local last CUDA error code.
 *  - Layouts (C order, densely packed): pos [n_blobs][3], force [n_rhs][n_blobs][3],
 *    vel [n_rhs][n_blobs][3] (or [n_rhs][row_count][3] for the *_rows calls).  Element
 *    type is double for RPY_PREC_F64 and float for RPY_PREC_F32_ACC64.  Blob order is
 *    preserved.  vel is overwritten.  All pointers must be aligned to their element type.
 *  - RPY_PREC_F64: every operation in IEEE double.  RPY_PREC_F32_ACC64: pair tensors in
 *    float, partial sums over at most 128 sources in float, running sums in double,
 *    output rounded to float once.
 *  - Device calls enqueue work on `cuda_stream` (a cudaStream_t passed as void*, NULL =
 *    the legacy default stream) and return without synchronising.  The workspace must
 *    stay untouched until that work has completed.
 *  - Errors are return codes only.  Nothing is enqueued when a code other than RPY_OK or
 *    RPY_ERR_CUDA is returned.  n_blobs == 0 (or row_count == 0) is RPY_OK and a no-op.
 *  - All kernels are compiled for sm_100a only; on any other device the first launch
 *    fails and RPY_ERR_CUDA is returned.  There is no CPU fallback.
 */
#ifndef RPY_MATVEC_H
#define RPY_MATVEC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    RPY_OK = 0,
    RPY_ERR_NULL = 1,       /* a required pointer is NULL                                   */
    RPY_ERR_ARG = 2,        /* n_blobs < 0, n_rhs < 1, bad row range, a or eta not finite > 0,
                               unknown precision, n_blobs above RPY_MAX_BLOBS               */
    RPY_ERR_ALIAS = 3,      /* d_vel overlaps d_pos, d_force or the workspace               */
    RPY_ERR_WORKSPACE = 4,  /* workspace smaller than rpy_matvec_workspace_bytes(), or not
                               256-byte aligned                                             */
    RPY_ERR_CUDA = 5        /* a CUDA runtime call failed; see rpy_last_cuda_error()        */
} rpy_status;

typedef enum {
    RPY_PREC_F64 = 0,       /* double in, double arithmetic, double out                     */
    RPY_PREC_F32_ACC64 = 1  /* float in, float pair arithmetic, double accumulation, float out */
} rpy_prec;

/* Largest n_blobs accepted (index arithmetic is 64-bit; the bound keeps N^2 work finite). */
#define RPY_MAX_BLOBS ((int64_t)1 << 26)

/* Bytes of device workspace the device calls need for (prec, n_blobs, n_rhs); 0 for
 * n_blobs <= 0 or n_rhs < 1.  Holds the packed source records (PAPER.md:75 composite
 * vectors r and lambda, rescaled by 1/a) and the double partial sums per source chunk.
 * The same size serves the *_rows calls with any row range. */
size_t rpy_matvec_workspace_bytes(rpy_prec prec, int64_t n_blobs, int n_rhs);

/* u = M lambda with the wall-corrected tensor, all rows.
 *   d_pos [n_blobs][3], d_force [n_rhs][n_blobs][3] : device, read only
 *   d_vel [n_rhs][n_blobs][3]                        : device, overwritten
 *   a, eta      : blob radius and viscosity, finite and > 0
 *   d_workspace : device, 256-byte aligned, >= rpy_matvec_workspace_bytes() bytes          */
rpy_status rpy_wall_matvec(rpy_prec prec, int64_t n_blobs, int n_rhs,
                           const void *d_pos, const void *d_force, void *d_vel,
                           double a, double eta,
                           void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* The same with the free-space RPY tensor, Eq. (9). */
rpy_status rpy_free_matvec(rpy_prec prec, int64_t n_blobs, int n_rhs,
                           const void *d_pos, const void *d_force, void *d_vel,
                           double a, double eta,
                           void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* Row-sharded forms: velocities of the target blobs row_begin .. row_begin+row_count-1
 * only, summed over ALL n_blobs sources (rows of M are independent, PAPER.md:562
 * "trivially parallelized"); this is the unit a multi-GPU caller gives each rank.
 *   d_vel [n_rhs][row_count][3].   0 <= row_begin, row_begin + row_count <= n_blobs.   */
rpy_status rpy_wall_matvec_rows(rpy_prec prec, int64_t n_blobs, int n_rhs,
                                int64_t row_begin, int64_t row_count,
                                const void *d_pos, const void *d_force, void *d_vel,
                                double a, double eta,
                                void *d_workspace, size_t workspace_bytes, void *cuda_stream);
rpy_status rpy_free_matvec_rows(rpy_prec prec, int64_t n_blobs, int n_rhs,
                                int64_t row_begin, int64_t row_count,
                                const void *d_pos, const void *d_force, void *d_vel,
                                double a, double eta,
                                void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* Work-sharded forms: one of n_shards PARTIAL products whose sum over shard = 0 .. n_shards-1 is
 * u = M lambda; the unit a multi-GPU caller gives each rank when it wants the symmetric kernel's
 * halved arithmetic on every GPU (it then adds the partial results with one all-reduce of
 * 3 n_rhs n_blobs doubles).  d_vel [n_rhs][n_blobs][3] is overwritten with the shard's contribution
 * to EVERY row and is DOUBLE on both paths: the cross-shard sum is part of the "fp64 accumulation" of
 * the fp32 path and must not round to float per shard (pos and force keep the path's type).
 * For n_rhs == 1 and n_blobs >= 1,152 a shard is a contiguous range of the tile
 * distances of the symmetric kernel (all distances cost the same, so shards are balanced); otherwise
 * it is a contiguous range of target rows of the plain kernel and the other rows are zero.
 * 0 <= shard < n_shards <= 4096.  Workspace: rpy_matvec_workspace_bytes().                        */
rpy_status rpy_wall_matvec_shard(rpy_prec prec, int64_t n_blobs, int n_rhs, int shard, int n_shards,
                                 const void *d_pos, const void *d_force, void *d_vel,
                                 double a, double eta,
                                 void *d_workspace, size_t workspace_bytes, void *cuda_stream);
rpy_status rpy_free_matvec_shard(rpy_prec prec, int64_t n_blobs, int n_rhs, int shard, int n_shards,
                                 const void *d_pos, const void *d_force, void *d_vel,
                                 double a, double eta,
                                 void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* Rectangular product: velocities at n_targets points that are not the sources,
 *   u_t = sum_{j < n_sources} M(r_t, r_j) lambda_j,
 * the flow-field evaluation of Appendix B: "the velocity that a freely-moving
 * tracer blob of a given size a' would have ... v(r) = sum_j M'(r - r_j) lambda'_j, where M' is the
 * blob-blob mobility for blobs of radius a'".  Targets and sources share the radius `a` (= a' in
 * the paper's use); a target that coincides with a source sees that source's self block.
 *   d_target_pos [n_targets][3], d_source_pos [n_sources][3], d_force [n_rhs][n_sources][3],
 *   d_vel [n_rhs][n_targets][3] (overwritten; all zero when n_sources == 0)
 *   d_workspace: >= rpy_matvec_rect_workspace_bytes(), 256-byte aligned.
 * Always the plain (bit-reproducible) all-pairs kernel.                                          */
size_t rpy_matvec_rect_workspace_bytes(rpy_prec prec, int64_t n_targets, int64_t n_sources, int n_rhs);
rpy_status rpy_wall_matvec_rect(rpy_prec prec, int64_t n_targets, int64_t n_sources, int n_rhs,
                                const void *d_target_pos, const void *d_source_pos, const void *d_force,
                                void *d_vel, double a, double eta,
                                void *d_workspace, size_t workspace_bytes, void *cuda_stream);
rpy_status rpy_free_matvec_rect(rpy_prec prec, int64_t n_targets, int64_t n_sources, int n_rhs,
                                const void *d_target_pos, const void *d_source_pos, const void *d_force,
                                void *d_vel, double a, double eta,
                                void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* Appendix B's source refinement: every blob i is replaced by n_sub small blobs at
 * r_i + template[s] (the template, in real lengths, is the caller's choice: the paper does not say
 * how the small blobs are placed) and its force is divided uniformly, lambda'_{i,s} = lambda_i / n_sub.
 *   d_pos [n_blobs][3], d_force [n_rhs][n_blobs][3], d_template [n_sub][3]  ->
 *   d_sub_pos [n_blobs * n_sub][3], d_sub_force [n_rhs][n_blobs * n_sub][3]   (sub-blob s of blob i at
 *   index i * n_sub + s).  1 <= n_sub <= 4096; n_blobs * n_sub <= RPY_MAX_BLOBS.                  */
rpy_status rpy_flow_subdivide(rpy_prec prec, int64_t n_blobs, int n_rhs, int n_sub,
                              const void *d_pos, const void *d_force, const void *d_template,
                              void *d_sub_pos, void *d_sub_force, void *cuda_stream);

/* Host-buffer forms ("only the positions of the blobs need to be communicated",
 * here positions and forces go up, velocities come back).
 *   h_pos, h_force, h_vel : HOST pointers, layouts as above
 *   d_scratch : device, 256-byte aligned, >= rpy_matvec_host_scratch_bytes() bytes
 * Copies the inputs host->device on `cuda_stream`, runs the matvec, copies the result
 * device->host and SYNCHRONISES the stream before returning, so h_vel is valid on return. */
size_t rpy_matvec_host_scratch_bytes(rpy_prec prec, int64_t n_blobs, int n_rhs);
rpy_status rpy_wall_matvec_host(rpy_prec prec, int64_t n_blobs, int n_rhs,
                                const void *h_pos, const void *h_force, void *h_vel,
                                double a, double eta,
                                void *d_scratch, size_t scratch_bytes, void *cuda_stream);
rpy_status rpy_free_matvec_host(rpy_prec prec, int64_t n_blobs, int n_rhs,
                                const void *h_pos, const void *h_force, void *h_vel,
                                double a, double eta,
                                void *d_scratch, size_t scratch_bytes, void *cuda_stream);

/* Counts blobs with z < zmin (e.g. zmin = a: blobs overlapping the wall, for which the
 * wall-corrected M is not positive definite).  d_count is a device
 * int64 that is overwritten (zeroed, then accumulated) in stream order. */
rpy_status rpy_wall_count_below(rpy_prec prec, int64_t n_blobs, const void *d_pos, double zmin,
                                int64_t *d_count, void *cuda_stream);

/* Launch geometry the all-pairs kernel would use for (prec, n_blobs, n_rhs, row_count).
 * Pure host arithmetic (no CUDA call); any output pointer may be NULL.
 *   *symmetric == 0: the plain kernel.  A CTA owns *targets_per_cta target rows and walks one of
 *     *n_source_chunks contiguous chunks of the sources in shared-memory tiles of *tile_sources.
 *   *symmetric == 1: the symmetric kernel (n_rhs == 1, all rows, n_blobs >= 1,152), which uses
 *     M_ij = M_ji^T to build every unordered pair's coefficients once.  Blobs are
 *     cut into tiles of *tile_sources (= *targets_per_cta: 128 below 50,000 blobs, else 256); a CTA owns one tile I and walks the
 *     tiles (I + d) mod n_tiles for one of *n_source_chunks chunks of the distances d = 0..n_tiles/2.
 *     Both halves of every CTA's work are accumulated with fp64 atomics into one double array, so the
 *     result is reproducible to rounding of the double sums (~1e-16 relative), not bit for bit; the plain
 *     kernel (and therefore every *_rows call and every n_rhs > 1 call) is bit-reproducible.
 *   *n_ctas: CTAs of the launch. */
rpy_status rpy_matvec_launch_plan(rpy_prec prec, int64_t n_blobs, int n_rhs, int64_t row_count,
                                  int *targets_per_cta, int *n_source_chunks,
                                  int *tile_sources, int64_t *n_ctas, int *symmetric);

const char *rpy_status_string(rpy_status s);

/* cudaError_t (as int) of the last RPY_ERR_CUDA returned on the calling thread, else 0. */
int rpy_last_cuda_error(void);

/* Version of this ABI (bumped on any signature change). */
int rpy_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RPY_MATVEC_H */
