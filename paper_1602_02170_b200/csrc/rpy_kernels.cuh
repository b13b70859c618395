// rpy_kernels.cuh -- the three kernels of the hot path:
//   prepack   O(N k): scale positions by 1/a and lay sources out as fixed-size records,
//   allpairs  O(N^2 k): the direct sum of Eq. (6),
//   finalise  O(N k): add the per-chunk double partials in fixed order, apply 1/(6 pi eta a).
//
// Source record ("group" = W consecutive sources, W = Lane::W):
//   S x[W], y[W], z[W], then for every right-hand side  S lx[W], ly[W], lz[W],
//   padded to a multiple of 16 bytes.  With W = 2 (packed float) one LDS.128 hands the
//   inner loop x and y of two sources already in the register-pair form FFMA2 wants.
// A staged tile is TILE_G consecutive records = one contiguous byte range, so it is
// fetched with ONE 1-D bulk async copy (cp.async.bulk, TMA engine) completing on an
// mbarrier; two buffers, the copy of tile t+1 overlaps the arithmetic on tile t.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "rpy_math.cuh"
#include "rpy_launch.cuh"

#ifndef RPY_SYM_UNROLL_F32
#define RPY_SYM_UNROLL_F32 4      // inner-loop unroll of the symmetric kernel (measured)
#endif
#ifndef RPY_SYM_UNROLL_F64
#define RPY_SYM_UNROLL_F64 4
#endif

#ifndef RPY_SYM_UNROLL_F32
#define RPY_SYM_UNROLL_F32 4
#endif
#ifndef RPY_SYM_UNROLL_F64
#define RPY_SYM_UNROLL_F64 4
#endif

namespace rpy {

template <class L, int K> struct RecLayout {
    using S = typename L::S;
    static constexpr int W = L::W;
    static constexpr int PER16 = 16 / (int)sizeof(S);
    static constexpr int RAW = (3 + 3 * K) * W;
    static constexpr int LEN = (RAW + PER16 - 1) / PER16 * PER16;   // scalars per record
    static constexpr int BYTES = LEN * (int)sizeof(S);
};

// ---------------------------------------------------------------------------- prepack
// One thread per (padded) source.  Sources beyond n_blobs are padding: position (0,0,1),
// zero force -- every coefficient stays finite and the contribution is exactly zero.
template <class L, int K>
__global__ void prepack_kernel(const typename L::S* __restrict__ pos,
                               const typename L::S* __restrict__ force,   // [K][n][3] of this RHS group
                               typename L::S* __restrict__ rec,
                               int64_t n_blobs, int64_t n_padded, int64_t force_rhs_stride,
                               double inv_a, double* __restrict__ zero, int64_t zero_count,
                               const int* __restrict__ skip)
{
    using S = typename L::S;
    using R = RecLayout<L, K>;
    pdl_enter();
    if (skip != nullptr && *skip != 0) return;      // a caller that enqueues ahead of a device-side decision (rpy_rigid.cu)
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_padded) return;
    // the symmetric kernel's atomic accumulator (3 doubles per blob) is cleared here: one launch less
    for (int64_t e = 3 * j; e < 3 * j + 3 && e < zero_count; ++e) zero[e] = 0.0;
    int64_t g = j / R::W;
    int l = (int)(j % R::W);
    S* r = rec + g * R::LEN;
    bool real = j < n_blobs;
    S x = real ? (S)((double)pos[3 * j + 0] * inv_a) : (S)0;
    S y = real ? (S)((double)pos[3 * j + 1] * inv_a) : (S)0;
    S z = real ? (S)((double)pos[3 * j + 2] * inv_a) : (S)1;
    r[0 * R::W + l] = x;
    r[1 * R::W + l] = y;
    r[2 * R::W + l] = z;
#pragma unroll
    for (int s = 0; s < K; ++s) {
        const S* f = force + (int64_t)s * force_rhs_stride + 3 * j;
        r[(3 + 3 * s + 0) * R::W + l] = real ? f[0] : (S)0;
        r[(3 + 3 * s + 1) * R::W + l] = real ? f[1] : (S)0;
        r[(3 + 3 * s + 2) * R::W + l] = real ? f[2] : (S)0;
    }
    if (l == 0) {
#pragma unroll
        for (int q = R::RAW; q < R::LEN; ++q) r[q] = (S)0;
    }
}

// Targets that are not sources (rectangular product, "Computing flow fields"):
// only the scaled coordinates are written, in the same record layout, so the all-pairs kernel
// reads its targets the same way in both cases.  Rows beyond n_targets are never read.
template <class L, int K>
__global__ void prepack_targets_kernel(const typename L::S* __restrict__ pos, typename L::S* __restrict__ rec,
                                       int64_t n_targets, double inv_a)
{
    using S = typename L::S;
    using R = RecLayout<L, K>;
    pdl_enter();
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_targets) return;
    S* r = rec + (j / R::W) * R::LEN;
    int l = (int)(j % R::W);
    r[0 * R::W + l] = (S)((double)pos[3 * j + 0] * inv_a);
    r[1 * R::W + l] = (S)((double)pos[3 * j + 1] * inv_a);
    r[2 * R::W + l] = (S)((double)pos[3 * j + 2] * inv_a);
}

// ---------------------------------------------------------------------------- mbarrier / bulk copy
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared (this CTA), completion counted in bytes on `bar`.
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------------------- all-pairs
// Grid: x = target tile (BLOCK*T targets), y = source chunk.  Each thread keeps T targets in
// registers (broadcast into every lane of V), walks the chunk's tiles from shared memory
// (every lane of a warp reads the same record: a broadcast, no bank conflict), and keeps
//   - float forms: per-target partial sums in V over FLUSH_G records (<= 128 sources), then
//     adds them into double running sums (the "fp64 accumulation" of north_star);
//   - double form: the running sums directly.
// Targets are read from `trec` (same record layout; equal to `rec` for the square product).
// Output: partial[chunk][s][row][3] in double (row relative to row_begin).
template <class L, int K, bool WALL, int T, int BLOCK, int TILE_G, int FLUSH_G, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
allpairs_kernel(const typename L::S* __restrict__ rec, const typename L::S* __restrict__ trec,
                double* __restrict__ partial,
                int64_t row_begin, int64_t row_count, int64_t n_tiles, int tiles_per_chunk,
                const int* __restrict__ skip)
{
    using V = typename L::V;
    using S = typename L::S;
    using R = RecLayout<L, K>;
    constexpr int W = L::W;
    constexpr bool IS_F64 = sizeof(S) == 8;
    constexpr uint32_t TILE_BYTES = (uint32_t)TILE_G * R::BYTES;
    static_assert(TILE_G % FLUSH_G == 0, "flush period must divide the tile");
    pdl_wait();
    if (skip != nullptr && *skip != 0) return;
    static_assert(TILE_BYTES % 16 == 0, "bulk copy size");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* const buf0 = smem_raw;      // buffer b lives at buf0 + b * TILE_BYTES
    __shared__ __align__(8) uint64_t full_bar[2];

    const int tid = threadIdx.x;
    const int64_t tile_lo = (int64_t)blockIdx.y * tiles_per_chunk;
    int64_t tile_hi = tile_lo + tiles_per_chunk;
    if (tile_hi > n_tiles) tile_hi = n_tiles;
    const int my_tiles = (int)(tile_hi - tile_lo);

    if (tid == 0) {
        mbar_init(&full_bar[0], 1);
        mbar_init(&full_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const unsigned char* gsrc = reinterpret_cast<const unsigned char*>(rec) + tile_lo * (int64_t)TILE_BYTES;
    if (tid == 0 && my_tiles > 0) {
        mbar_expect_tx(&full_bar[0], TILE_BYTES);
        bulk_g2s(buf0, gsrc, TILE_BYTES, &full_bar[0]);
    }

    // targets of this thread: rows row_begin + (blockIdx.x*BLOCK*T + t*BLOCK + tid); rows past
    // the end recompute the last row and are not stored.
    V xi[T], yi[T], zi[T], zi2[T];
    int64_t row[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        row[t] = (int64_t)blockIdx.x * (BLOCK * T) + t * BLOCK + tid;
        int64_t i = row_begin + (row[t] < row_count ? row[t] : row_count - 1);
        const S* r = trec + (i / W) * R::LEN + (i % W);      // trec == rec unless targets differ from sources
        xi[t] = L::bc((double)r[0 * W]);
        yi[t] = L::bc((double)r[1 * W]);
        zi[t] = L::bc((double)r[2 * W]);
        zi2[t] = L::bc(2.0 * (double)r[2 * W]);
    }

    double dacc[IS_F64 ? 1 : T][IS_F64 ? 1 : K][3];
    V acc[T][K][3];
#pragma unroll
    for (int t = 0; t < T; ++t)
#pragma unroll
        for (int s = 0; s < K; ++s)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                acc[t][s][c] = L::bc(0.0);
                if constexpr (!IS_F64) dacc[t][s][c] = 0.0;
            }

    for (int it = 0; it < my_tiles; ++it) {
        const int b = it & 1;
        // every thread is done with buffer b^1 (read in iteration it-1) before it is refilled
        __syncthreads();
        if (tid == 0 && it + 1 < my_tiles) {
            mbar_expect_tx(&full_bar[b ^ 1], TILE_BYTES);
            bulk_g2s(buf0 + (b ^ 1) * TILE_BYTES, gsrc + (int64_t)(it + 1) * TILE_BYTES, TILE_BYTES, &full_bar[b ^ 1]);
        }
        mbar_wait(&full_bar[b], (uint32_t)((it >> 1) & 1));
        const S* tile = reinterpret_cast<const S*>(buf0 + b * TILE_BYTES);

#pragma unroll 1
        for (int g0 = 0; g0 < TILE_G; g0 += FLUSH_G) {
#pragma unroll 2
            for (int g = g0; g < g0 + FLUSH_G; ++g) {
                const V* r = reinterpret_cast<const V*>(tile + g * R::LEN);
                V xj = r[0], yj = r[1], zj = r[2];
                V lam[K][3];
#pragma unroll
                for (int s = 0; s < K; ++s) {
                    lam[s][0] = r[3 + 3 * s + 0];
                    lam[s][1] = r[3 + 3 * s + 1];
                    lam[s][2] = r[3 + 3 * s + 2];
                }
                // phase 1 (every pair): separation and the r > 2a scalars of Eq. (9)
                PairCoef<V> c[T];
                PairPre<V> pre[T];
                bool near = false;
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    pair_pre<L, WALL>(xi[t], yi[t], zi[t], xj, yj, zj, c[t], pre[t]);
                    near = near || L::any_le(pre[t].r2, 4.0);
                }
                // phase 2 (rare, warp-uniform): some lane has an overlapping pair (r <= 2a) or r = 0
                if (__any_sync(0xffffffffu, near)) {
#pragma unroll
                    for (int t = 0; t < T; ++t) rpy_near_fixup<L, WALL>(pre[t].r2, pre[t].n1, pre[t].f, pre[t].G);
                }
                // phase 3 (every pair): wall scalars and the product with lambda_j
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    pair_post<L, WALL>(zi2[t], zj, pre[t], c[t]);
#pragma unroll
                    for (int s = 0; s < K; ++s)
                        pair_apply<L, WALL>(c[t], lam[s][0], lam[s][1], lam[s][2],
                                            acc[t][s][0], acc[t][s][1], acc[t][s][2]);
                }
            }
            if constexpr (!IS_F64) {
#pragma unroll
                for (int t = 0; t < T; ++t)
#pragma unroll
                    for (int s = 0; s < K; ++s)
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            dacc[t][s][c] += L::hsum(acc[t][s][c]);
                            acc[t][s][c] = L::bc(0.0);
                        }
            }
        }
    }

    double* out = partial + (int64_t)blockIdx.y * K * row_count * 3;
#pragma unroll
    for (int t = 0; t < T; ++t) {
        if (row[t] < row_count) {
#pragma unroll
            for (int s = 0; s < K; ++s)
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    if constexpr (IS_F64) out[((int64_t)s * row_count + row[t]) * 3 + c] = L::hsum(acc[t][s][c]);
                    else                  out[((int64_t)s * row_count + row[t]) * 3 + c] = dacc[t][s][c];
        }
    }
}

// ---------------------------------------------------------------------------- all-pairs, symmetric
// Uses M_ij = M_ji^T (M is symmetric by construction of Eq. (7)): the five pair
// coefficients of the unordered pair {i, j} are built ONCE and applied twice,
//   u_i += M_ij lambda_j   (forward,    accumulators stay with the thread that owns target i),
//   u_j += M_ij^T lambda_i (transposed, accumulators TRAVEL with the source),
// which costs 44 + 2*10 FP-pipe operations per unordered pair instead of 2*(44 + 10).
//
// Decomposition.  Blobs are cut into tiles of TS = BLOCK*T; tile I meets tile J = (I + d) mod nt
// for d = 0 .. nt/2: every unordered tile pair exactly once (for even nt the distance nt/2 is
// taken by I < nt/2 only), every I the same amount of work.  Grid: x = I, y = chunk of the d range.
// d = 0 is the diagonal tile: all TS x TS ordered pairs are walked forward with the transposed
// application switched off (lambda_i := 0 there).
//
// Inside a tile pair each thread owns T targets of I.  A warp walks J in sub-tiles of 32 source
// groups: at step s lane l reads group (s + l) mod 32 from shared memory (each lane a different
// 48-byte record: bank-conflict-free) and holds that group's transposed
// accumulators, which it hands to lane l-1 by one warp shuffle per component after the step.
// After 32 steps every group has met all 32*T targets of the warp and is back in its home lane,
// which adds the float partial (<= 32*T terms) into the double array `gacc` with one fp64 atomic
// per component: the order of those atomics is the only non-deterministic part of the result.
// The four warps start on different sub-tiles so they never flush the same addresses together.
template <class V> __device__ __forceinline__ V shfl_from(V v, int src_lane);
template <> __device__ __forceinline__ double shfl_from<double>(double v, int src_lane) { return __shfl_sync(0xffffffffu, v, src_lane); }
template <> __device__ __forceinline__ float shfl_from<float>(float v, int src_lane) { return __shfl_sync(0xffffffffu, v, src_lane); }
template <> __device__ __forceinline__ float2 shfl_from<float2>(float2 v, int src_lane)
{
    return make_float2(__shfl_sync(0xffffffffu, v.x, src_lane), __shfl_sync(0xffffffffu, v.y, src_lane));
}
template <class V> __device__ __forceinline__ double lane_elem(V v, int w);
template <> __device__ __forceinline__ double lane_elem<double>(double v, int) { return v; }
template <> __device__ __forceinline__ double lane_elem<float>(float v, int) { return (double)v; }
template <> __device__ __forceinline__ double lane_elem<float2>(float2 v, int w) { return (double)(w ? v.y : v.x); }

template <class L, bool WALL, int T, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
allpairs_sym_kernel(const typename L::S* __restrict__ rec, double* __restrict__ gacc,
                    int64_t n_blobs, int nt, int d_per_chunk, int d_begin, int d_end, int split,
                    const int* __restrict__ skip)
{
    using V = typename L::V;
    using S = typename L::S;
    using R = RecLayout<L, 1>;
    constexpr int W = L::W;
    constexpr bool IS_F64 = sizeof(S) == 8;
    constexpr int TS = BLOCK * T;                  // blobs per tile
    pdl_wait();
    if (skip != nullptr && *skip != 0) return;
    constexpr int TILE_G = TS / W;                 // records per tile
    constexpr int NSUB = TILE_G / 32;              // sub-tiles of 32 records
    constexpr int NWARP = BLOCK / 32;
    constexpr int kUnroll = IS_F64 ? RPY_SYM_UNROLL_F64 : RPY_SYM_UNROLL_F32;
    constexpr uint32_t TILE_BYTES = (uint32_t)TILE_G * R::BYTES;
    static_assert(TILE_G % 32 == 0 && R::LEN * sizeof(S) == 48, "record geometry");
    // Small problems do not fill the chip with one CTA per tile pair (N = 2,000: 136 tile pairs of 128 blobs for 888
    // resident CTAs): the host may cut every tile pair into `split` parts (grid z); this CTA then meets only the sub-tiles
    // p_lo .. p_lo + cnt - 1 of each tile J (and stages only those), with all of its own targets.
    const int cnt = NSUB / split;                  // sub-tiles per tile for this CTA (split divides NSUB)
    const int p_lo = (int)blockIdx.z * cnt;
    const uint32_t part_bytes = (uint32_t)cnt * 32u * R::BYTES;
    const int64_t part_off = (int64_t)p_lo * 32 * R::BYTES;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* const buf0 = smem_raw;
    __shared__ __align__(8) uint64_t full_bar[2];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int I = blockIdx.x;
    const int D = nt / 2;                          // largest tile distance
    // this launch covers the tile distances d_begin .. d_end-1 (all of 0 .. D unless the work is
    // sharded over several GPUs: every distance costs the same, so a shard is a range of distances)
    const int d_lo = d_begin + blockIdx.y * d_per_chunk;
    int d_hi = d_lo + d_per_chunk;
    if (d_hi > d_end) d_hi = d_end;
    if ((nt & 1) == 0 && d_hi == D + 1 && I >= D && D > 0) d_hi = D;   // distance nt/2: lower half only
    if (nt == 1) d_hi = d_lo == 0 ? 1 : 0;
    const int my_tiles = d_hi - d_lo;

    if (tid == 0) {
        mbar_init(&full_bar[0], 1);
        mbar_init(&full_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const unsigned char* gbase = reinterpret_cast<const unsigned char*>(rec);
    auto tile_of = [&](int it) { int J = I + d_lo + it; return J >= nt ? J - nt : J; };
    if (tid == 0 && my_tiles > 0) {
        mbar_expect_tx(&full_bar[0], part_bytes);
        bulk_g2s(buf0, gbase + (int64_t)tile_of(0) * TILE_BYTES + part_off, part_bytes, &full_bar[0]);
    }

    V xi[T], yi[T], zi[T], zi2[T], li[T][3];
    int64_t row[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        row[t] = (int64_t)I * TS + t * BLOCK + tid;            // < n_padded: a real record (maybe padding)
        const S* r = rec + (row[t] / W) * R::LEN + (row[t] % W);
        xi[t] = L::bc((double)r[0 * W]);
        yi[t] = L::bc((double)r[1 * W]);
        zi[t] = L::bc((double)r[2 * W]);
        zi2[t] = L::bc(2.0 * (double)r[2 * W]);
        li[t][0] = L::bc((double)r[3 * W]);
        li[t][1] = L::bc((double)r[4 * W]);
        li[t][2] = L::bc((double)r[5 * W]);
    }

    double dacc[IS_F64 ? 1 : T][3];
    V acc[T][3];
#pragma unroll
    for (int t = 0; t < T; ++t)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            acc[t][c] = L::bc(0.0);
            if constexpr (!IS_F64) dacc[t][c] = 0.0;
        }

    for (int it = 0; it < my_tiles; ++it) {
        const int b = it & 1;
        __syncthreads();                                       // buffer b^1 is free again
        if (tid == 0 && it + 1 < my_tiles) {
            mbar_expect_tx(&full_bar[b ^ 1], part_bytes);
            bulk_g2s(buf0 + (b ^ 1) * TILE_BYTES, gbase + (int64_t)tile_of(it + 1) * TILE_BYTES + part_off, part_bytes, &full_bar[b ^ 1]);
        }
        mbar_wait(&full_bar[b], (uint32_t)((it >> 1) & 1));
        const S* tile = reinterpret_cast<const S*>(buf0 + b * TILE_BYTES);     // holds sub-tiles p_lo .. p_lo + cnt - 1 of J
        const int J = tile_of(it);
        const bool diagonal = (d_lo + it) == 0;
        V lt[T][3];                                            // lambda_i as seen by the transposed application
#pragma unroll
        for (int t = 0; t < T; ++t)
#pragma unroll
            for (int c = 0; c < 3; ++c) lt[t][c] = diagonal ? L::bc(0.0) : li[t][c];

#pragma unroll 1
        for (int p = 0; p < cnt; ++p) {
            // the warps start on different sub-tiles (when the CTA has several) so that they do not flush the same
            // addresses together; ql = index inside the staged part, q = index inside the tile
            const int ql = (p + warp * (NSUB / NWARP > 0 ? NSUB / NWARP : 1)) % cnt;
            const int q = p_lo + ql;
            const S* sub = tile + (ql * 32) * R::LEN;
            V uj[3] = {L::bc(0.0), L::bc(0.0), L::bc(0.0)};
#pragma unroll kUnroll              // measured (cfg 3, end of round 2): fp32 896 / 912 / 908 G pairs/s with 2 / 4 / 8; fp64 391 / 391 / 397
            for (int s = 0; s < 32; ++s) {
                const int g = (s + lane) & 31;
                const V* r = reinterpret_cast<const V*>(sub + g * R::LEN);
                V xj = r[0], yj = r[1], zj = r[2];
                V lj0 = r[3], lj1 = r[4], lj2 = r[5];
                PairCoef<V> c[T];
                PairPre<V> pre[T];
                bool near = false;
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    pair_pre<L, WALL>(xi[t], yi[t], zi[t], xj, yj, zj, c[t], pre[t]);
                    near = near || L::any_le(pre[t].r2, 4.0);
                }
                if (__any_sync(0xffffffffu, near)) {
#pragma unroll
                    for (int t = 0; t < T; ++t) rpy_near_fixup<L, WALL>(pre[t].r2, pre[t].n1, pre[t].f, pre[t].G);
                }
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    pair_post<L, WALL>(zi2[t], zj, pre[t], c[t]);
                    // forward (u_i += M_ij lambda_j) and transposed (u_j += M_ij^T lambda_i) side by side
                    pair_apply_both<L, WALL>(c[t], lj0, lj1, lj2, acc[t][0], acc[t][1], acc[t][2],
                                             lt[t][0], lt[t][1], lt[t][2], uj[0], uj[1], uj[2]);
                }
                const int from = (lane + 1) & 31;              // the lane that just served group g + 1
                uj[0] = shfl_from<V>(uj[0], from);
                uj[1] = shfl_from<V>(uj[1], from);
                uj[2] = shfl_from<V>(uj[2], from);
            }
            // home again: lane holds the sum over this warp's 32*T targets for record q*32 + lane
            if (!diagonal) {
#pragma unroll
                for (int w = 0; w < W; ++w) {
                    int64_t j = (int64_t)J * TS + (int64_t)(q * 32 + lane) * W + w;
                    if (j < n_blobs) {
                        atomicAdd(gacc + j * 3 + 0, lane_elem<V>(uj[0], w));
                        atomicAdd(gacc + j * 3 + 1, lane_elem<V>(uj[1], w));
                        atomicAdd(gacc + j * 3 + 2, lane_elem<V>(uj[2], w));
                    }
                }
            }
            if constexpr (!IS_F64) {
#pragma unroll
                for (int t = 0; t < T; ++t)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        dacc[t][c] += L::hsum(acc[t][c]);
                        acc[t][c] = L::bc(0.0);
                    }
            }
        }
    }

    // the forward half of this CTA's chunk joins the transposed halves in the one double accumulator: no per-chunk
    // slices to write and to add up afterwards (at N = 15,000 they were 61 x 360 KB per product)
#pragma unroll
    for (int t = 0; t < T; ++t) {
        if (row[t] < n_blobs && my_tiles > 0) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
                if constexpr (IS_F64) atomicAdd(gacc + row[t] * 3 + c, L::hsum(acc[t][c]));
                else                  atomicAdd(gacc + row[t] * 3 + c, dacc[t][c]);
        }
    }
}

// ---------------------------------------------------------------------------- finalise
// vel[s][row][c] = scale * sum_{chunk} partial[chunk][s][row][c], chunks added in a fixed order
// (deterministic), one thread per output element.
template <class S>
__global__ void finalise_kernel(const double* __restrict__ partial, S* __restrict__ vel,
                                int64_t per_chunk /* = K*row_count*3 */, int n_chunks,
                                int64_t row_count3, int64_t vel_rhs_stride, double scale,
                                const int* __restrict__ skip)
{
    pdl_enter();
    int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= per_chunk || (skip != nullptr && *skip != 0)) return;
    // four interleaved running sums (fixed assignment chunk -> sum, fixed final order): the loads of
    // different chunks do not wait on one another
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int c = 0;
    for (; c + 4 <= n_chunks; c += 4) {
        s0 += partial[(int64_t)c * per_chunk + e];
        s1 += partial[(int64_t)(c + 1) * per_chunk + e];
        s2 += partial[(int64_t)(c + 2) * per_chunk + e];
        s3 += partial[(int64_t)(c + 3) * per_chunk + e];
    }
    for (; c < n_chunks; ++c) s0 += partial[(int64_t)c * per_chunk + e];
    const double sum = (s0 + s1) + (s2 + s3);
    int64_t s = e / row_count3, q = e % row_count3;
    vel[s * vel_rhs_stride + q] = (S)(sum * scale);
}

// Appendix B: blob i -> n_sub small blobs at r_i + template[s], force lambda_i / n_sub.
template <class S>
__global__ void subdivide_kernel(const S* __restrict__ pos, const S* __restrict__ force, const S* __restrict__ tmpl,
                                 S* __restrict__ sub_pos, S* __restrict__ sub_force, int64_t n_blobs, int n_rhs, int n_sub)
{
    const int64_t total = n_blobs * n_sub;
    const S div = (S)n_sub;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = e / n_sub;
        const int s = (int)(e % n_sub);
#pragma unroll
        for (int c = 0; c < 3; ++c) sub_pos[3 * e + c] = pos[3 * i + c] + tmpl[3 * s + c];
        for (int r = 0; r < n_rhs; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                sub_force[((int64_t)r * total + e) * 3 + c] = force[((int64_t)r * n_blobs + i) * 3 + c] / div;
    }
}

template <class S>
__global__ void count_below_kernel(const S* __restrict__ pos, int64_t n, double zmin,
                                   unsigned long long* __restrict__ count)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool below = i < n && (double)pos[3 * i + 2] < zmin;
    unsigned m = __ballot_sync(0xffffffffu, below);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(count, (unsigned long long)__popc(m));
}

}  // namespace rpy
