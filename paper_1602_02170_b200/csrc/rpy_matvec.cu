// rpy_matvec.cu -- host side of the C ABI declared in include/rpy_matvec.h: argument checks,
// launch planning, and the prepack -> all-pairs -> finalise launch sequence.  No allocation,
// no synchronisation (except the *_host forms), no state.  sm_100a only.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/rpy_matvec.h"
#include "rpy_kernels.cuh"
#include "rpy_internal.h"

#ifndef RPY_SYM_MINB_F32
#define RPY_SYM_MINB_F32 3
#endif
#ifndef RPY_SYM_MINB_F64
#define RPY_SYM_MINB_F64 4
#endif

namespace {

thread_local int g_last_cuda_error = 0;

constexpr int kAbiVersion = 5;
constexpr int kNumSMs = 148;             // B200: 2 dies x 74 SMs
constexpr int kTargetCtas = kNumSMs * 64;  // no source chunking beyond this many CTAs
constexpr int kSymTargetCtas = kNumSMs * 256;   // the symmetric kernel's chunks of tile distances aim at this many
constexpr int kMaxChunks = 64;
constexpr int kBlock = 128;
constexpr int kMaxT = 2;
constexpr size_t kAlign = 256;
constexpr int kSymTile = kBlock * 2;       // blobs per tile of the symmetric kernel (T = 2)
#ifndef RPY_SYM_MIN_BLOBS
#define RPY_SYM_MIN_BLOBS 1152
#endif
constexpr int64_t kSymMinBlobs = RPY_SYM_MIN_BLOBS;   // below this the plain kernel is used (too few tile pairs to fill the chip)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Per (precision, K) kernel shape.  TILE_G records per staged tile, FLUSH_G records per
// float->double flush (W*FLUSH_G <= 128 sources, the bound stated in the header).
template <class L, int K> struct Shape;
template <int K> struct Shape<rpy::Lane<float2>, K> {
    static constexpr int TILE_G = 64, FLUSH_G = 64, MINB = (K >= 4 ? 2 : 4);
};
template <int K> struct Shape<rpy::Lane<double>, K> {
    static constexpr int TILE_G = 64, FLUSH_G = 64, MINB = (K >= 4 ? 1 : 2);
};

struct Plan {
    int T;                 // targets per thread
    int targets_per_cta;
    int tile_sources;      // W * TILE_G
    int64_t n_padded;      // sources incl. padding
    int64_t n_tiles;
    int tiles_per_chunk;
    int n_chunks;
    int64_t n_target_tiles;
};

inline int tile_sources_of(rpy_prec prec) { return prec == RPY_PREC_F64 ? 64 : 128; }
inline size_t elem_size(rpy_prec prec) { return prec == RPY_PREC_F64 ? 8 : 4; }

// scalars per record, mirrors rpy::RecLayout
inline size_t record_bytes(rpy_prec prec, int K)
{
    int W = prec == RPY_PREC_F64 ? 1 : 2;
    int per16 = 16 / (int)elem_size(prec);
    int raw = (3 + 3 * K) * W;
    return (size_t)((raw + per16 - 1) / per16 * per16) * elem_size(prec);
}

// Two targets per thread once there are enough rows to fill the chip that way (K >= 4 already
// holds 3K accumulators per target: one target per thread there).
inline int choose_T(int K, int64_t rows)
{
    return (K <= 2 && rows >= (int64_t)kNumSMs * kBlock * 2 * 2) ? 2 : 1;
}

// The source range is cut into n_chunks so that the CTAs spread evenly over the 148 SMs.  The
// kernel is ALU-bound and every CTA does the same work, so the time is set by the SM that is
// handed the most CTAs, m = ceil(CTAs / 148), and by how long the last CTAs run on a partly empty
// SM.  Measured on B200 (cfg 2, cfg 3, both precisions, 4..64 chunks): throughput rises
// monotonically with the CTA count up to ~64 CTAs per SM (cfg 3 fp32: 496 G pairs/s at 18 CTAs
// per SM, 519 at 64+; the fixed cost of a CTA is far below one tile), so: aim for kTargetCtas,
// and among the chunk counts in the upper half of the allowed range take the one with the least
// quantisation loss tiles_per_chunk * m.
Plan make_plan(rpy_prec prec, int64_t n, int K, int64_t rows)
{
    Plan p;
    p.tile_sources = tile_sources_of(prec);
    p.n_padded = (n + p.tile_sources - 1) / p.tile_sources * p.tile_sources;
    p.n_tiles = p.n_padded / p.tile_sources;
    p.T = choose_T(K, rows);
    p.targets_per_cta = kBlock * p.T;
    p.n_target_tiles = (rows + p.targets_per_cta - 1) / p.targets_per_cta;
    int64_t c_max = p.n_target_tiles > 0 ? (kTargetCtas + p.n_target_tiles - 1) / p.n_target_tiles : 1;
    if (c_max > kMaxChunks) c_max = kMaxChunks;
    if (c_max > p.n_tiles) c_max = p.n_tiles;
    if (c_max < 1) c_max = 1;
    int64_t best_cost = -1;
    p.tiles_per_chunk = (int)p.n_tiles; p.n_chunks = 1;
    for (int64_t want = (c_max + 1) / 2; want <= c_max; ++want) {
        int64_t tpc = (p.n_tiles + want - 1) / want;
        int64_t nch = (p.n_tiles + tpc - 1) / tpc;
        int64_t per_sm = (p.n_target_tiles * nch + kNumSMs - 1) / kNumSMs;
        int64_t cost = tpc * per_sm;
        if (best_cost < 0 || cost <= best_cost) {
            best_cost = cost; p.tiles_per_chunk = (int)tpc; p.n_chunks = (int)nch;
        }
    }
    return p;
}

inline int group_k(int remaining) { return remaining >= 8 ? 8 : remaining >= 4 ? 4 : remaining >= 2 ? 2 : 1; }

size_t records_bytes(rpy_prec prec, int64_t n, int K)
{
    int ts = kSymTile;                       // a multiple of every kernel's tile (64 / 128 / 256 sources)
    int64_t n_padded = (n + ts - 1) / ts * ts;
    int W = prec == RPY_PREC_F64 ? 1 : 2;
    return align_up((size_t)(n_padded / W) * record_bytes(prec, K), kAlign);
}

// n_chunks * rows <= kTargetCtas * kBlock * kMaxT + rows  (n_chunks <= kTargetCtas / n_target_tiles + 1)
// and n_chunks <= n_tiles, rows <= n.
// `rows` target rows against `n` sources (rows <= n for the square product; any ratio for the
// rectangular one).
size_t partial_bytes_bound(rpy_prec prec, int64_t n, int K, int64_t rows)
{
    int ts = tile_sources_of(prec);
    int64_t n_tiles = (n + ts - 1) / ts;
    int64_t a = (int64_t)kTargetCtas * kBlock * (K <= 2 ? kMaxT : 1) + 2 * rows;   // (the symmetric path needs one slice)
    int64_t b = n_tiles * rows;
    return align_up((size_t)(a < b ? a : b) * (size_t)K * 3 * sizeof(double), kAlign);
}

size_t workspace_bytes(rpy_prec prec, int64_t n, int n_rhs)
{
    if (n <= 0 || n_rhs < 1) return 0;
    int K = group_k(n_rhs);
    return records_bytes(prec, n, K) + partial_bytes_bound(prec, n, K, n);
}

// rectangular product: source records, target records, partials
size_t rect_workspace_bytes(rpy_prec prec, int64_t n_targets, int64_t n_sources, int n_rhs)
{
    if (n_targets <= 0 || n_sources <= 0 || n_rhs < 1) return 0;
    int K = group_k(n_rhs);
    return records_bytes(prec, n_sources, K) + records_bytes(prec, n_targets, K) +
           partial_bytes_bound(prec, n_sources, K, n_targets);
}

inline rpy_status cuda_fail(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    return RPY_ERR_CUDA;
}

inline bool overlaps(const void* p, size_t pn, const void* q, size_t qn)
{
    uintptr_t a = (uintptr_t)p, b = (uintptr_t)q;
    return pn && qn && a < b + qn && b < a + pn;
}

template <class L, int K, bool WALL, int T>
auto allpairs_fn()
{
    using Sh = Shape<L, K>;
    return rpy::allpairs_kernel<L, K, WALL, T, kBlock, Sh::TILE_G, Sh::FLUSH_G, Sh::MINB>;
}
template <class L, int K> constexpr size_t allpairs_smem() { return 2 * (size_t)Shape<L, K>::TILE_G * rpy::RecLayout<L, K>::BYTES; }

template <class L, int K, bool WALL, int T>
cudaError_t launch_allpairs(const Plan& p, const typename L::S* rec, const typename L::S* trec, double* partial,
                            int64_t row_begin, int64_t rows, cudaStream_t st, const int* skip)
{
    dim3 grid((unsigned)p.n_target_tiles, (unsigned)p.n_chunks);
    return rpy::launch_pdl(allpairs_fn<L, K, WALL, T>(), grid, dim3(kBlock), allpairs_smem<L, K>(), st,
                           rec, trec, partial, row_begin, rows, p.n_tiles, p.tiles_per_chunk, skip);
}

// Symmetric path (rpy::allpairs_sym_kernel): one right-hand side, all rows, enough tiles.
struct SymPlan { int nt; int d_per_chunk; int n_chunks; int64_t n_padded; int d_begin; int d_end; int tile; int split; };

#ifndef RPY_SYM_SPLIT_BELOW_CTAS_PER_SM
#define RPY_SYM_SPLIT_BELOW_CTAS_PER_SM 6
#endif
#ifndef RPY_SYM_SMALL_BELOW
#define RPY_SYM_SMALL_BELOW 50000      // below this many blobs the symmetric kernel runs with 128-blob tiles (measured crossover)
#endif
struct Shard { int index; int count; };        // {0, 1}: the whole product

// What varies between the entry points that share run_group.
struct Opts {
    Shard sh{0, 1};
    int64_t vel_stride3 = -1;       // elements between right-hand sides of vel (-1: 3 rows)
    int64_t force_stride3 = -1;     // the same for force (-1: 3 n)
    bool vel_f64 = false;           // vel is double whatever the path (partial products of a shard)
    const int* skip = nullptr;      // device flag: non-zero turns every kernel of the call into a no-op
    rpy::PartialSums* partials = nullptr;   // non-null: finalise is left to the caller, who gets the slices
    bool chain_in = false;          // the call's first kernel may be scheduled under the kernel before it in the stream
                                    // (programmatic dependent launch): a caller that chains its own kernels (the solver)
};

inline bool use_symmetric(int64_t n, int K, int64_t row_begin, int64_t rows)
{
    return K == 1 && row_begin == 0 && rows == n && n >= kSymMinBlobs;
}

// max_split: 32-record sub-tiles of a 128-blob tile (2 with two blobs per record, 4 with one)
SymPlan make_sym_plan(int64_t n, int max_split, Shard sh = Shard{0, 1})
{
    SymPlan p;
    // Tiles of 256 blobs (128 threads x 2 targets) once there are enough of them to fill the chip several
    // times over; 128-blob tiles (64 threads x 2) below that: four times as many, four times smaller CTAs.
    // (64-blob tiles, one warp per CTA, were measured too: a gain only at N = 3,584 ... 3,900)
    p.tile = n < RPY_SYM_SMALL_BELOW ? kSymTile / 2 : kSymTile;
    p.n_padded = (n + kSymTile - 1) / kSymTile * kSymTile;       // records are padded to 256 either way
    p.nt = (int)((n + p.tile - 1) / p.tile);
    const int all = p.nt / 2 + 1;                              // tile distances 0 .. nt/2
    p.d_begin = (int)((int64_t)all * sh.index / sh.count);     // shard = a contiguous range of distances
    p.d_end = (int)((int64_t)all * (sh.index + 1) / sh.count);
    int count = p.d_end - p.d_begin;
    if (count < 1) count = 1;                                  // an empty shard still launches (and writes zeros)
    // many short CTAs: measured (cfg 3 / cfg 4, fp32, G pairs/s) 148 x 64 CTAs 914.6 / 909.9, x 128 915.3 / 918.3,
    // x 256 918.7 / 921.8, x 512 920.1 / 921.8
    int64_t want = (kSymTargetCtas + p.nt - 1) / p.nt;
    if (want > count) want = count;
    if (want < 1) want = 1;
    p.d_per_chunk = (int)((count + want - 1) / want);
    p.n_chunks = (count + p.d_per_chunk - 1) / p.d_per_chunk;
    // Small problems: one CTA per tile pair does not fill the chip (N = 2,000: 136 tile pairs for 148 x 6 resident CTAs of
    // 64 threads): cut every tile pair into two halves of its source tile (grid z).  Past that point the halves only add
    // set-up and flush work (measured: N = 3,584 29.2 -> 24.0 us, N >= 4,000 within 2 %).
    p.split = 1;
#ifndef RPY_SYM_NO_SPLIT
    if (p.tile == kSymTile / 2 && p.d_per_chunk == 1)
        while (p.split < max_split && (int64_t)p.nt * p.n_chunks * p.split <= (int64_t)kNumSMs * RPY_SYM_SPLIT_BELOW_CTAS_PER_SM)
            p.split *= 2;
#endif
    return p;
}

template <class L> struct SymShape;
template <> struct SymShape<rpy::Lane<float2>> { static constexpr int MINB = RPY_SYM_MINB_F32; };
template <> struct SymShape<rpy::Lane<double>> { static constexpr int MINB = RPY_SYM_MINB_F64; };

template <class L>
cudaError_t launch_sym(bool wall, const SymPlan& p, const typename L::S* rec, double* gacc,
                       int64_t n, cudaStream_t st, const int* skip)
{
    constexpr int MINB = SymShape<L>::MINB;
    dim3 grid((unsigned)p.nt, (unsigned)p.n_chunks, (unsigned)p.split);
    if (p.tile == kSymTile) {
        size_t smem = 2 * (size_t)(kSymTile / L::W) * rpy::RecLayout<L, 1>::BYTES;
        if (wall) return rpy::launch_pdl(rpy::allpairs_sym_kernel<L, true, 2, kBlock, MINB>, grid, dim3(kBlock), smem, st,
                                         rec, gacc, n, p.nt, p.d_per_chunk, p.d_begin, p.d_end, p.split, skip);
        return rpy::launch_pdl(rpy::allpairs_sym_kernel<L, false, 2, kBlock, MINB>, grid, dim3(kBlock), smem, st,
                               rec, gacc, n, p.nt, p.d_per_chunk, p.d_begin, p.d_end, p.split, skip);
    }
    constexpr int B2 = kBlock / 2;
    size_t smem = 2 * (size_t)(kSymTile / 2 / L::W) * rpy::RecLayout<L, 1>::BYTES;
    if (wall) return rpy::launch_pdl(rpy::allpairs_sym_kernel<L, true, 2, B2, 2 * MINB>, grid, dim3(B2), smem, st,
                                     rec, gacc, n, p.nt, p.d_per_chunk, p.d_begin, p.d_end, p.split, skip);
    return rpy::launch_pdl(rpy::allpairs_sym_kernel<L, false, 2, B2, 2 * MINB>, grid, dim3(B2), smem, st,
                           rec, gacc, n, p.nt, p.d_per_chunk, p.d_begin, p.d_end, p.split, skip);
}

template <class L, int K>
cudaError_t run_group(bool wall, int64_t n, int64_t row_begin, int64_t rows,
                      const typename L::S* pos, const typename L::S* force, void* vel,
                      double a, double eta, unsigned char* ws, cudaStream_t st, void* const* ev,
                      const typename L::S* tpos /* targets of the rectangular product, else nullptr */,
                      const Opts& o)
{
    const Shard sh = o.sh;
    const int64_t vel_stride3 = o.vel_stride3, force_stride3 = o.force_stride3;
    const bool vel_f64 = o.vel_f64;
    const int* skip = o.skip;
    using S = typename L::S;
    S* rec = reinterpret_cast<S*>(ws);
    rpy_prec prec = sizeof(S) == 8 ? RPY_PREC_F64 : RPY_PREC_F32_ACC64;
    size_t at = records_bytes(prec, n, K);
    const S* trec = rec;
    if (tpos) {                                    // rows = n_targets, row_begin = 0
        S* tr = reinterpret_cast<S*>(ws + at);
        at += records_bytes(prec, rows, K);
        int threads = 256;
        cudaError_t e0 = rpy::launch_chain(o.chain_in, rpy::prepack_targets_kernel<L, K>, dim3((unsigned)((rows + threads - 1) / threads)), dim3(threads), 0, st,
                                         tpos, tr, rows, 1.0 / a);
        if (e0 != cudaSuccess) return e0;
        trec = tr;
    }
    double* partial = reinterpret_cast<double*>(ws + at);
    const bool sym = !tpos && use_symmetric(n, K, row_begin, rows);
    const Plan p = make_plan(prec, n, K, rows);
    const SymPlan sp = make_sym_plan(n, kSymTile / 2 / L::W / 32, sh);
    const int64_t n_padded = sym ? sp.n_padded : p.n_padded;
    cudaError_t e;
    int n_slices = p.n_chunks;
    // symmetric kernel: ONE slice, which receives both halves of every CTA's work through fp64 atomics
    double* gacc = sym ? partial : nullptr;
    {
        int threads = 256;
        int64_t blocks = (n_padded + threads - 1) / threads;
        e = rpy::launch_chain(o.chain_in || tpos != nullptr, rpy::prepack_kernel<L, K>, dim3((unsigned)blocks), dim3(threads), 0, st,
                            pos, force, rec, n, n_padded, force_stride3, 1.0 / a, gacc, sym ? n * 3 : (int64_t)0, skip);
        if (e != cudaSuccess) return e;
    }
    if (sym) {
        if (ev && (e = cudaEventRecord(static_cast<cudaEvent_t>(ev[1]), st)) != cudaSuccess) return e;
        if constexpr (K == 1) e = launch_sym<L>(wall, sp, rec, gacc, n, st, skip);
        else e = cudaErrorInvalidValue;
        n_slices = 1;
    } else {
        if (ev && (e = cudaEventRecord(static_cast<cudaEvent_t>(ev[1]), st)) != cudaSuccess) return e;
        constexpr int T2 = K <= 2 ? 2 : 1;     // choose_T never asks for T = 2 when K > 2
        if (wall) e = p.T == 2 ? launch_allpairs<L, K, true, T2>(p, rec, trec, partial, row_begin, rows, st, skip)
                               : launch_allpairs<L, K, true, 1>(p, rec, trec, partial, row_begin, rows, st, skip);
        else      e = p.T == 2 ? launch_allpairs<L, K, false, T2>(p, rec, trec, partial, row_begin, rows, st, skip)
                               : launch_allpairs<L, K, false, 1>(p, rec, trec, partial, row_begin, rows, st, skip);
    }
    if (e != cudaSuccess) return e;
    if (ev && (e = cudaEventRecord(static_cast<cudaEvent_t>(ev[2]), st)) != cudaSuccess) return e;
    {
        int64_t per_chunk = (int64_t)K * rows * 3;
        int threads = 256;
        int64_t blocks = (per_chunk + threads - 1) / threads;
        const double PI = 3.14159265358979323846;
        const double scale = 1.0 / (6.0 * PI * eta * a);
        if (o.partials) {                           // the caller adds the slices itself (fused into its next kernel)
            o.partials->partial = partial; o.partials->n_slices = n_slices;
            o.partials->per_chunk = per_chunk; o.partials->scale = scale;
            return cudaSuccess;
        }
        (void)vel_stride3;
        if (vel_f64) e = rpy::launch_pdl(rpy::finalise_kernel<double>, dim3((unsigned)blocks), dim3(threads), 0, st,
                                         partial, static_cast<double*>(vel), per_chunk, n_slices, rows * 3, vel_stride3, scale, skip);
        else         e = rpy::launch_pdl(rpy::finalise_kernel<S>, dim3((unsigned)blocks), dim3(threads), 0, st,
                                         partial, static_cast<S*>(vel), per_chunk, n_slices, rows * 3, vel_stride3, scale, skip);
    }
    return e;
}

template <class L>
cudaError_t run_all_groups(bool wall, int64_t n, int n_rhs, int64_t row_begin, int64_t rows,
                           const void* d_pos, const void* d_force, void* d_vel,
                           double a, double eta, void* ws, cudaStream_t st, void* const* ev,
                           const void* d_tpos = nullptr, Opts o = Opts{})
{
    using S = typename L::S;
    cudaError_t ee;
    if (ev && (ee = cudaEventRecord(static_cast<cudaEvent_t>(ev[0]), st)) != cudaSuccess) return ee;
    const S* pos = static_cast<const S*>(d_pos);
    const S* tp = static_cast<const S*>(d_tpos);
    if (o.vel_stride3 < 0) o.vel_stride3 = rows * 3;
    if (o.force_stride3 < 0) o.force_stride3 = n * 3;
    int done = 0;
    while (done < n_rhs) {
        int K = group_k(n_rhs - done);
        const S* force = static_cast<const S*>(d_force) + (int64_t)done * o.force_stride3;
        void* vel = d_vel ? static_cast<unsigned char*>(d_vel) + (size_t)done * o.vel_stride3 * (o.vel_f64 ? sizeof(double) : sizeof(S)) : nullptr;
        unsigned char* w = static_cast<unsigned char*>(ws);
        void* const* ev1 = done == 0 ? ev : nullptr;
        cudaError_t e;
        switch (K) {
            case 8: e = run_group<L, 8>(wall, n, row_begin, rows, pos, force, vel, a, eta, w, st, ev1, tp, o); break;
            case 4: e = run_group<L, 4>(wall, n, row_begin, rows, pos, force, vel, a, eta, w, st, ev1, tp, o); break;
            case 2: e = run_group<L, 2>(wall, n, row_begin, rows, pos, force, vel, a, eta, w, st, ev1, tp, o); break;
            default: e = run_group<L, 1>(wall, n, row_begin, rows, pos, force, vel, a, eta, w, st, ev1, tp, o); break;
        }
        if (e != cudaSuccess) return e;
        done += K;
    }
    if (ev && (ee = cudaEventRecord(static_cast<cudaEvent_t>(ev[3]), st)) != cudaSuccess) return ee;
    return cudaSuccess;
}

rpy_status matvec_rows(bool wall, rpy_prec prec, int64_t n, int n_rhs, int64_t row_begin, int64_t rows,
                       const void* d_pos, const void* d_force, void* d_vel, double a, double eta,
                       void* ws, size_t ws_bytes, void* stream, void* const* ev = nullptr)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n < 0 || n > RPY_MAX_BLOBS || n_rhs < 1) return RPY_ERR_ARG;
    if (row_begin < 0 || rows < 0 || row_begin > n || rows > n - row_begin) return RPY_ERR_ARG;
    if (!(a > 0.0) || !(eta > 0.0) || !isfinite(a) || !isfinite(eta)) return RPY_ERR_ARG;
    if (n == 0 || rows == 0) return RPY_OK;
    if (!d_pos || !d_force || !d_vel || !ws) return RPY_ERR_NULL;
    size_t es = elem_size(prec);
    size_t pos_b = (size_t)n * 3 * es, force_b = pos_b * (size_t)n_rhs, vel_b = (size_t)rows * 3 * es * (size_t)n_rhs;
    size_t need = workspace_bytes(prec, n, n_rhs);
    if (ws_bytes < need || ((uintptr_t)ws % kAlign) != 0) return RPY_ERR_WORKSPACE;
    if (overlaps(d_vel, vel_b, d_pos, pos_b) || overlaps(d_vel, vel_b, d_force, force_b) ||
        overlaps(d_vel, vel_b, ws, need))
        return RPY_ERR_ALIAS;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e = prec == RPY_PREC_F64
        ? run_all_groups<rpy::Lane<double>>(wall, n, n_rhs, row_begin, rows, d_pos, d_force, d_vel, a, eta, ws, st, ev)
        : run_all_groups<rpy::Lane<float2>>(wall, n, n_rhs, row_begin, rows, d_pos, d_force, d_vel, a, eta, ws, st, ev);
    if (e != cudaSuccess) return cuda_fail(e);
    return RPY_OK;
}

// One of n_shards partial products whose SUM over the shards is u = M lambda (a multi-GPU caller adds
// them with an all-reduce).  With one right-hand side and enough blobs the shard is a range of tile
// distances of the symmetric kernel (M_ij = M_ji^T): every shard does 1/n_shards of the
// unordered pairs and produces contributions to ALL rows.  Otherwise the shard is a range of target
// rows of the plain kernel and the other rows of its output are zero.
rpy_status matvec_shard(bool wall, rpy_prec prec, int64_t n, int n_rhs, int shard, int n_shards, const void* d_pos,
                        const void* d_force, void* d_vel, double a, double eta, void* ws, size_t ws_bytes, void* stream)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n < 0 || n > RPY_MAX_BLOBS || n_rhs < 1 || n_shards < 1 || n_shards > 4096 || shard < 0 || shard >= n_shards) return RPY_ERR_ARG;
    if (!(a > 0.0) || !(eta > 0.0) || !isfinite(a) || !isfinite(eta)) return RPY_ERR_ARG;
    if (n == 0) return RPY_OK;
    if (!d_pos || !d_force || !d_vel || !ws) return RPY_ERR_NULL;
    size_t es = elem_size(prec);
    size_t pos_b = (size_t)n * 3 * es, force_b = pos_b * (size_t)n_rhs;
    size_t vel_b = (size_t)n * 3 * sizeof(double) * (size_t)n_rhs;       // partial velocities are double on both paths
    size_t need = workspace_bytes(prec, n, n_rhs);
    if (ws_bytes < need || ((uintptr_t)ws % kAlign) != 0) return RPY_ERR_WORKSPACE;
    if (overlaps(d_vel, vel_b, d_pos, pos_b) || overlaps(d_vel, vel_b, d_force, force_b) || overlaps(d_vel, vel_b, ws, need))
        return RPY_ERR_ALIAS;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    if (n_rhs == 1 && use_symmetric(n, 1, 0, n)) {
        Opts o; o.sh = Shard{shard, n_shards}; o.vel_f64 = true;
        e = prec == RPY_PREC_F64
            ? run_all_groups<rpy::Lane<double>>(wall, n, 1, 0, n, d_pos, d_force, d_vel, a, eta, ws, st, nullptr, nullptr, o)
            : run_all_groups<rpy::Lane<float2>>(wall, n, 1, 0, n, d_pos, d_force, d_vel, a, eta, ws, st, nullptr, nullptr, o);
    } else {
        const int64_t r0 = n * shard / n_shards, r1 = n * (shard + 1) / n_shards;
        if ((e = cudaMemsetAsync(d_vel, 0, vel_b, st)) != cudaSuccess) return cuda_fail(e);
        if (r1 == r0) return RPY_OK;
        void* out = static_cast<unsigned char*>(d_vel) + (size_t)r0 * 3 * sizeof(double);
        // rows r0..r1-1 by the plain kernel (never the symmetric one: row_begin/rows are not the whole range,
        // or n is below the symmetric threshold), written in place of the full-length layout
        Opts o; o.vel_stride3 = n * 3; o.vel_f64 = true;
        e = prec == RPY_PREC_F64
            ? run_all_groups<rpy::Lane<double>>(wall, n, n_rhs, r0, r1 - r0, d_pos, d_force, out, a, eta, ws, st, nullptr, nullptr, o)
            : run_all_groups<rpy::Lane<float2>>(wall, n, n_rhs, r0, r1 - r0, d_pos, d_force, out, a, eta, ws, st, nullptr, nullptr, o);
    }
    if (e != cudaSuccess) return cuda_fail(e);
    return RPY_OK;
}

// u_t = sum_j M(r_t, r_j) lambda_j for targets that are not the sources.
rpy_status matvec_rect(bool wall, rpy_prec prec, int64_t nt, int64_t ns, int n_rhs, const void* d_tpos,
                       const void* d_spos, const void* d_force, void* d_vel, double a, double eta,
                       void* ws, size_t ws_bytes, void* stream)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (nt < 0 || ns < 0 || nt > RPY_MAX_BLOBS || ns > RPY_MAX_BLOBS || n_rhs < 1) return RPY_ERR_ARG;
    if (!(a > 0.0) || !(eta > 0.0) || !isfinite(a) || !isfinite(eta)) return RPY_ERR_ARG;
    if (nt == 0) return RPY_OK;
    if (!d_vel) return RPY_ERR_NULL;
    size_t es = elem_size(prec);
    size_t vel_b = (size_t)nt * 3 * es * (size_t)n_rhs;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (ns == 0) {                                  // empty sum
        cudaError_t e = cudaMemsetAsync(d_vel, 0, vel_b, st);
        return e == cudaSuccess ? RPY_OK : cuda_fail(e);
    }
    if (!d_tpos || !d_spos || !d_force || !ws) return RPY_ERR_NULL;
    size_t need = rect_workspace_bytes(prec, nt, ns, n_rhs);
    if (ws_bytes < need || ((uintptr_t)ws % kAlign) != 0) return RPY_ERR_WORKSPACE;
    size_t spos_b = (size_t)ns * 3 * es;
    if (overlaps(d_vel, vel_b, d_tpos, (size_t)nt * 3 * es) || overlaps(d_vel, vel_b, d_spos, spos_b) ||
        overlaps(d_vel, vel_b, d_force, spos_b * (size_t)n_rhs) || overlaps(d_vel, vel_b, ws, need))
        return RPY_ERR_ALIAS;
    cudaError_t e = prec == RPY_PREC_F64
        ? run_all_groups<rpy::Lane<double>>(wall, ns, n_rhs, 0, nt, d_spos, d_force, d_vel, a, eta, ws, st, nullptr, d_tpos)
        : run_all_groups<rpy::Lane<float2>>(wall, ns, n_rhs, 0, nt, d_spos, d_force, d_vel, a, eta, ws, st, nullptr, d_tpos);
    if (e != cudaSuccess) return cuda_fail(e);
    return RPY_OK;
}

size_t host_scratch_bytes(rpy_prec prec, int64_t n, int n_rhs)
{
    if (n <= 0 || n_rhs < 1) return 0;
    size_t es = elem_size(prec);
    size_t pos_b = align_up((size_t)n * 3 * es, kAlign);
    size_t f_b = align_up((size_t)n * 3 * es * (size_t)n_rhs, kAlign);
    return pos_b + 2 * f_b + workspace_bytes(prec, n, n_rhs);
}

rpy_status matvec_host(bool wall, rpy_prec prec, int64_t n, int n_rhs, const void* h_pos, const void* h_force,
                       void* h_vel, double a, double eta, void* d_scratch, size_t scratch_bytes, void* stream)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n < 0 || n > RPY_MAX_BLOBS || n_rhs < 1) return RPY_ERR_ARG;
    if (!(a > 0.0) || !(eta > 0.0) || !isfinite(a) || !isfinite(eta)) return RPY_ERR_ARG;
    if (n == 0) return RPY_OK;
    if (!h_pos || !h_force || !h_vel || !d_scratch) return RPY_ERR_NULL;
    if (scratch_bytes < host_scratch_bytes(prec, n, n_rhs) || ((uintptr_t)d_scratch % kAlign) != 0)
        return RPY_ERR_WORKSPACE;
    size_t es = elem_size(prec);
    size_t pos_raw = (size_t)n * 3 * es, f_raw = pos_raw * (size_t)n_rhs;
    size_t pos_b = align_up(pos_raw, kAlign), f_b = align_up(f_raw, kAlign);
    unsigned char* base = static_cast<unsigned char*>(d_scratch);
    void* d_pos = base;
    void* d_force = base + pos_b;
    void* d_vel = base + pos_b + f_b;
    void* ws = base + pos_b + 2 * f_b;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaMemcpyAsync(d_pos, h_pos, pos_raw, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaMemcpyAsync(d_force, h_force, f_raw, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e);
    rpy_status s = matvec_rows(wall, prec, n, n_rhs, 0, n, d_pos, d_force, d_vel, a, eta, ws,
                               workspace_bytes(prec, n, n_rhs), stream);
    if (s != RPY_OK) return s;
    e = cudaMemcpyAsync(h_vel, d_vel, f_raw, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e);
    return RPY_OK;
}

}  // namespace

namespace rpy {
rpy_status set_cuda_error(cudaError_t e) { return cuda_fail(e); }

rpy_status matvec_phases(bool wall, rpy_prec prec, int64_t n_blobs, int n_rhs, const void* d_pos, const void* d_force,
                         void* d_vel, double a, double eta, void* ws, size_t ws_bytes, void* stream, void* const* events4)
{
    if (!events4 || !events4[0] || !events4[1] || !events4[2] || !events4[3]) return RPY_ERR_NULL;
    if (n_blobs < 1) return RPY_ERR_ARG;
    return matvec_rows(wall, prec, n_blobs, n_rhs, 0, n_blobs, d_pos, d_force, d_vel, a, eta, ws, ws_bytes, stream, events4);
}

rpy_status matvec_strided(bool wall, rpy_prec prec, int64_t n, int n_rhs, const void* d_pos, const void* d_force,
                          int64_t force_stride3, void* d_vel, int64_t vel_stride3, double a, double eta,
                          void* ws, size_t ws_bytes, cudaStream_t st, const int* d_skip, PartialSums* partials,
                          int shard, int n_shards, bool vel_f64)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n < 1 || n > RPY_MAX_BLOBS || n_rhs < 1 || force_stride3 < 3 * n) return RPY_ERR_ARG;
    if (n_shards < 1 || shard < 0 || shard >= n_shards) return RPY_ERR_ARG;
    if (partials) {                               // one right-hand-side group, so that its slices outlive the call
        if (n_rhs != group_k(n_rhs)) return RPY_ERR_ARG;
    } else if (!d_vel || vel_stride3 < 3 * n) return RPY_ERR_ARG;
    if (n_shards > 1 && !(n_rhs == 1 && use_symmetric(n, 1, 0, n))) return RPY_ERR_ARG;   // shards of the symmetric kernel only
    if (!d_pos || !d_force || !ws) return RPY_ERR_NULL;
    if (ws_bytes < workspace_bytes(prec, n, n_rhs) || ((uintptr_t)ws % kAlign) != 0) return RPY_ERR_WORKSPACE;
    Opts o;
    o.vel_stride3 = partials ? 3 * n : vel_stride3; o.force_stride3 = force_stride3;
    o.skip = d_skip; o.partials = partials; o.sh = Shard{shard, n_shards}; o.vel_f64 = vel_f64;
    o.chain_in = true;                            // internal callers launch their own kernels chained as well
    cudaError_t e = prec == RPY_PREC_F64
        ? run_all_groups<rpy::Lane<double>>(wall, n, n_rhs, 0, n, d_pos, d_force, d_vel, a, eta, ws, st, nullptr, nullptr, o)
        : run_all_groups<rpy::Lane<float2>>(wall, n, n_rhs, 0, n, d_pos, d_force, d_vel, a, eta, ws, st, nullptr, nullptr, o);
    if (e != cudaSuccess) return cuda_fail(e);
    return RPY_OK;
}

bool matvec_shardable(int64_t n) { return use_symmetric(n, 1, 0, n); }
}  // namespace rpy

extern "C" {

size_t rpy_matvec_workspace_bytes(rpy_prec prec, int64_t n_blobs, int n_rhs)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return 0;
    if (n_blobs > RPY_MAX_BLOBS) return 0;
    return workspace_bytes(prec, n_blobs, n_rhs);
}

rpy_status rpy_wall_matvec(rpy_prec prec, int64_t n_blobs, int n_rhs, const void* d_pos, const void* d_force,
                           void* d_vel, double a, double eta, void* d_workspace, size_t workspace_bytes_,
                           void* cuda_stream)
{
    return matvec_rows(true, prec, n_blobs, n_rhs, 0, n_blobs < 0 ? 0 : n_blobs, d_pos, d_force, d_vel, a, eta,
                       d_workspace, workspace_bytes_, cuda_stream);
}

rpy_status rpy_free_matvec(rpy_prec prec, int64_t n_blobs, int n_rhs, const void* d_pos, const void* d_force,
                           void* d_vel, double a, double eta, void* d_workspace, size_t workspace_bytes_,
                           void* cuda_stream)
{
    return matvec_rows(false, prec, n_blobs, n_rhs, 0, n_blobs < 0 ? 0 : n_blobs, d_pos, d_force, d_vel, a, eta,
                       d_workspace, workspace_bytes_, cuda_stream);
}

rpy_status rpy_wall_matvec_rows(rpy_prec prec, int64_t n_blobs, int n_rhs, int64_t row_begin, int64_t row_count,
                                const void* d_pos, const void* d_force, void* d_vel, double a, double eta,
                                void* d_workspace, size_t workspace_bytes_, void* cuda_stream)
{
    if (n_blobs < 0) return RPY_ERR_ARG;
    return matvec_rows(true, prec, n_blobs, n_rhs, row_begin, row_count, d_pos, d_force, d_vel, a, eta,
                       d_workspace, workspace_bytes_, cuda_stream);
}

rpy_status rpy_free_matvec_rows(rpy_prec prec, int64_t n_blobs, int n_rhs, int64_t row_begin, int64_t row_count,
                                const void* d_pos, const void* d_force, void* d_vel, double a, double eta,
                                void* d_workspace, size_t workspace_bytes_, void* cuda_stream)
{
    if (n_blobs < 0) return RPY_ERR_ARG;
    return matvec_rows(false, prec, n_blobs, n_rhs, row_begin, row_count, d_pos, d_force, d_vel, a, eta,
                       d_workspace, workspace_bytes_, cuda_stream);
}

rpy_status rpy_wall_matvec_shard(rpy_prec prec, int64_t n_blobs, int n_rhs, int shard, int n_shards, const void* d_pos,
                                 const void* d_force, void* d_vel, double a, double eta, void* d_workspace,
                                 size_t workspace_bytes_, void* cuda_stream)
{
    return matvec_shard(true, prec, n_blobs, n_rhs, shard, n_shards, d_pos, d_force, d_vel, a, eta, d_workspace, workspace_bytes_, cuda_stream);
}

rpy_status rpy_free_matvec_shard(rpy_prec prec, int64_t n_blobs, int n_rhs, int shard, int n_shards, const void* d_pos,
                                 const void* d_force, void* d_vel, double a, double eta, void* d_workspace,
                                 size_t workspace_bytes_, void* cuda_stream)
{
    return matvec_shard(false, prec, n_blobs, n_rhs, shard, n_shards, d_pos, d_force, d_vel, a, eta, d_workspace, workspace_bytes_, cuda_stream);
}

size_t rpy_matvec_rect_workspace_bytes(rpy_prec prec, int64_t n_targets, int64_t n_sources, int n_rhs)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return 0;
    if (n_targets > RPY_MAX_BLOBS || n_sources > RPY_MAX_BLOBS) return 0;
    return rect_workspace_bytes(prec, n_targets, n_sources, n_rhs);
}

rpy_status rpy_wall_matvec_rect(rpy_prec prec, int64_t n_targets, int64_t n_sources, int n_rhs,
                                const void* d_target_pos, const void* d_source_pos, const void* d_force,
                                void* d_vel, double a, double eta, void* d_workspace, size_t workspace_bytes_,
                                void* cuda_stream)
{
    return matvec_rect(true, prec, n_targets, n_sources, n_rhs, d_target_pos, d_source_pos, d_force, d_vel, a, eta,
                       d_workspace, workspace_bytes_, cuda_stream);
}

rpy_status rpy_free_matvec_rect(rpy_prec prec, int64_t n_targets, int64_t n_sources, int n_rhs,
                                const void* d_target_pos, const void* d_source_pos, const void* d_force,
                                void* d_vel, double a, double eta, void* d_workspace, size_t workspace_bytes_,
                                void* cuda_stream)
{
    return matvec_rect(false, prec, n_targets, n_sources, n_rhs, d_target_pos, d_source_pos, d_force, d_vel, a, eta,
                       d_workspace, workspace_bytes_, cuda_stream);
}

rpy_status rpy_flow_subdivide(rpy_prec prec, int64_t n_blobs, int n_rhs, int n_sub, const void* d_pos,
                              const void* d_force, const void* d_template, void* d_sub_pos, void* d_sub_force,
                              void* cuda_stream)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n_blobs < 0 || n_rhs < 1 || n_sub < 1 || n_sub > 4096 || n_blobs * (int64_t)n_sub > RPY_MAX_BLOBS) return RPY_ERR_ARG;
    if (n_blobs == 0) return RPY_OK;
    if (!d_pos || !d_force || !d_template || !d_sub_pos || !d_sub_force) return RPY_ERR_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int64_t total = n_blobs * n_sub;
    unsigned blocks = (unsigned)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
    if (prec == RPY_PREC_F64)
        rpy::subdivide_kernel<double><<<blocks, 256, 0, st>>>((const double*)d_pos, (const double*)d_force, (const double*)d_template,
                                                             (double*)d_sub_pos, (double*)d_sub_force, n_blobs, n_rhs, n_sub);
    else
        rpy::subdivide_kernel<float><<<blocks, 256, 0, st>>>((const float*)d_pos, (const float*)d_force, (const float*)d_template,
                                                            (float*)d_sub_pos, (float*)d_sub_force, n_blobs, n_rhs, n_sub);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return RPY_OK;
}

size_t rpy_matvec_host_scratch_bytes(rpy_prec prec, int64_t n_blobs, int n_rhs)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return 0;
    if (n_blobs > RPY_MAX_BLOBS) return 0;
    return host_scratch_bytes(prec, n_blobs, n_rhs);
}

rpy_status rpy_wall_matvec_host(rpy_prec prec, int64_t n_blobs, int n_rhs, const void* h_pos, const void* h_force,
                                void* h_vel, double a, double eta, void* d_scratch, size_t scratch_bytes,
                                void* cuda_stream)
{
    return matvec_host(true, prec, n_blobs, n_rhs, h_pos, h_force, h_vel, a, eta, d_scratch, scratch_bytes, cuda_stream);
}

rpy_status rpy_free_matvec_host(rpy_prec prec, int64_t n_blobs, int n_rhs, const void* h_pos, const void* h_force,
                                void* h_vel, double a, double eta, void* d_scratch, size_t scratch_bytes,
                                void* cuda_stream)
{
    return matvec_host(false, prec, n_blobs, n_rhs, h_pos, h_force, h_vel, a, eta, d_scratch, scratch_bytes, cuda_stream);
}

rpy_status rpy_wall_count_below(rpy_prec prec, int64_t n_blobs, const void* d_pos, double zmin, int64_t* d_count,
                                void* cuda_stream)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n_blobs < 0 || n_blobs > RPY_MAX_BLOBS || isnan(zmin)) return RPY_ERR_ARG;
    if (!d_count) return RPY_ERR_NULL;
    if (n_blobs > 0 && !d_pos) return RPY_ERR_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t e = cudaMemsetAsync(d_count, 0, sizeof(int64_t), st);
    if (e != cudaSuccess) return cuda_fail(e);
    if (n_blobs == 0) return RPY_OK;
    int threads = 256;
    unsigned blocks = (unsigned)((n_blobs + threads - 1) / threads);
    auto* cnt = reinterpret_cast<unsigned long long*>(d_count);
    if (prec == RPY_PREC_F64)
        rpy::count_below_kernel<double><<<blocks, threads, 0, st>>>(static_cast<const double*>(d_pos), n_blobs, zmin, cnt);
    else
        rpy::count_below_kernel<float><<<blocks, threads, 0, st>>>(static_cast<const float*>(d_pos), n_blobs, zmin, cnt);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return RPY_OK;
}

rpy_status rpy_matvec_launch_plan(rpy_prec prec, int64_t n_blobs, int n_rhs, int64_t row_count,
                                  int* targets_per_cta, int* n_source_chunks, int* tile_sources, int64_t* n_ctas,
                                  int* symmetric)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n_blobs < 0 || n_blobs > RPY_MAX_BLOBS || n_rhs < 1 || row_count < 0 || row_count > n_blobs) return RPY_ERR_ARG;
    const int K = group_k(n_rhs);
    if (use_symmetric(n_blobs, K, 0, row_count) && n_rhs == 1) {
        SymPlan sp = make_sym_plan(n_blobs, prec == RPY_PREC_F64 ? 4 : 2);
        if (targets_per_cta) *targets_per_cta = sp.tile;
        if (n_source_chunks) *n_source_chunks = sp.n_chunks;
        if (tile_sources) *tile_sources = sp.tile;
        if (n_ctas) *n_ctas = (int64_t)sp.nt * sp.n_chunks * sp.split;
        if (symmetric) *symmetric = 1;
        return RPY_OK;
    }
    Plan p = make_plan(prec, n_blobs, K, row_count);
    if (targets_per_cta) *targets_per_cta = p.targets_per_cta;
    if (n_source_chunks) *n_source_chunks = p.n_chunks;
    if (tile_sources) *tile_sources = p.tile_sources;
    if (n_ctas) *n_ctas = p.n_target_tiles * p.n_chunks;
    if (symmetric) *symmetric = 0;
    return RPY_OK;
}

const char* rpy_status_string(rpy_status s)
{
    switch (s) {
        case RPY_OK: return "RPY_OK";
        case RPY_ERR_NULL: return "RPY_ERR_NULL: a required pointer is NULL";
        case RPY_ERR_ARG: return "RPY_ERR_ARG: invalid size, range, precision, radius or viscosity";
        case RPY_ERR_ALIAS: return "RPY_ERR_ALIAS: output overlaps an input or the workspace";
        case RPY_ERR_WORKSPACE: return "RPY_ERR_WORKSPACE: workspace too small or misaligned";
        case RPY_ERR_CUDA: return "RPY_ERR_CUDA: a CUDA runtime call failed (rpy_last_cuda_error)";
    }
    return "unknown rpy_status";
}

int rpy_last_cuda_error(void) { return g_last_cuda_error; }
int rpy_abi_version(void) { return kAbiVersion; }

}  // extern "C"
