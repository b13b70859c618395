// rpy_rigid.cu -- the rigid-multiblob layer of include/rpy_rigid.h: K, K^T (Eqs. (2)-(3), (10)),
// the block-diagonal preconditioner of Eqs. (17)-(19) (dense per-body M^(pp), Cholesky, N~_pp) and
// right-preconditioned GMRES on the saddle-point system (11).  arXiv:1602.02170 Section II
// (PAPER.md:79-84, 154-252).  sm_100a only; no allocation, no state.
//
// Kernels:
//   k_apply / kt_apply / saddle_tail     one warp per body; O(N_b)
//   precond_build             one CTA per body: dense M^(pp) from the same pair arithmetic as the
//                             matvec (rpy_math.cuh, double lanes), in-place Cholesky, explicit inverse
//                             from the factor, Y = M^-1 K, N~ = (K^T Y)^-1
//   precond_apply             one warp per body: symmetric matrix-vector product + 6x6 work
//   dots / update / normalise (+ Hessenberg) / combine     the Krylov vector operations of GMRES
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/rpy_rigid.h"
#include "rpy_math.cuh"
#include "rpy_launch.cuh"
#include "rpy_internal.h"

namespace {

constexpr size_t kAlign = 256;
constexpr int kSmemBodyM = 162;            // largest 3*blobs whose matrix is factorised in shared memory
constexpr int kBuildThreads = 256;
constexpr int64_t kMagic = 0x52505952494744LL;   // "RPYRIGD"
constexpr int kVecBlocks = 296;            // CTAs of the Krylov vector kernels: 2 per SM
constexpr int kVecThreads = 256;
constexpr int kScal = 8;                   // doubles of scalar state per right-hand side of the solve
constexpr int kSnapBytes = 128;            // one snapshot of the solve's state for the host (16 + 8 * RPY_RIGID_MAX_BATCH <= 128)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline rpy_status st_of(int s) { return static_cast<rpy_status>(s); }

// ------------------------------------------------------------------ K and K^T
// (K U)_i = u_p + omega_p x (r_i - q_p), Eq. (2).
__global__ void k_apply_kernel(const double* __restrict__ pos, const double* __restrict__ q,
                               const int64_t* __restrict__ offsets, const double* __restrict__ U,
                               double alpha, double beta, double* __restrict__ out, int64_t n_bodies,
                               int64_t u_stride, int64_t out_stride /* between right-hand sides (blockIdx.y) */)
{
    const int64_t p = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (p >= n_bodies) return;
    U += (int64_t)blockIdx.y * u_stride; out += (int64_t)blockIdx.y * out_stride;
    const double ux = U[6 * p + 0], uy = U[6 * p + 1], uz = U[6 * p + 2];
    const double wx = U[6 * p + 3], wy = U[6 * p + 4], wz = U[6 * p + 5];
    const double qx = q[3 * p + 0], qy = q[3 * p + 1], qz = q[3 * p + 2];
    for (int64_t i = offsets[p] + lane; i < offsets[p + 1]; i += 32) {
        const double dx = pos[3 * i + 0] - qx, dy = pos[3 * i + 1] - qy, dz = pos[3 * i + 2] - qz;
        const double vx = ux + (wy * dz - wz * dy);
        const double vy = uy + (wz * dx - wx * dz);
        const double vz = uz + (wx * dy - wy * dx);
        if (beta == 0.0) {
            out[3 * i + 0] = alpha * vx; out[3 * i + 1] = alpha * vy; out[3 * i + 2] = alpha * vz;
        } else {
            out[3 * i + 0] = beta * out[3 * i + 0] + alpha * vx;
            out[3 * i + 1] = beta * out[3 * i + 1] + alpha * vy;
            out[3 * i + 2] = beta * out[3 * i + 2] + alpha * vz;
        }
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// f_p = sum lambda_i, tau_p = sum (r_i - q_p) x lambda_i, Eq. (10).
__global__ void kt_apply_kernel(const double* __restrict__ pos, const double* __restrict__ q,
                                const int64_t* __restrict__ offsets, const double* __restrict__ lam,
                                double alpha, double beta, double* __restrict__ out, int64_t n_bodies,
                                int64_t lam_stride, int64_t out_stride /* between right-hand sides (blockIdx.y) */)
{
    const int64_t p = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (p >= n_bodies) return;
    lam += (int64_t)blockIdx.y * lam_stride; out += (int64_t)blockIdx.y * out_stride;
    const double qx = q[3 * p + 0], qy = q[3 * p + 1], qz = q[3 * p + 2];
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int64_t i = offsets[p] + lane; i < offsets[p + 1]; i += 32) {
        const double dx = pos[3 * i + 0] - qx, dy = pos[3 * i + 1] - qy, dz = pos[3 * i + 2] - qz;
        const double lx = lam[3 * i + 0], ly = lam[3 * i + 1], lz = lam[3 * i + 2];
        s[0] += lx; s[1] += ly; s[2] += lz;
        s[3] += dy * lz - dz * ly;
        s[4] += dz * lx - dx * lz;
        s[5] += dx * ly - dy * lx;
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) s[c] = warp_sum(s[c]);
    if (lane < 6) {
        double v = s[0];
#pragma unroll
        for (int c = 1; c < 6; ++c) if (lane == c) v = s[c];
        out[6 * p + lane] = (beta == 0.0 ? 0.0 : beta * out[6 * p + lane]) + alpha * v;
    }
}

// scale * (sum of the product's per-slice partial sums) for output element e of right-hand side blockIdx.y, the
// slices added in the order of the product's own finalise kernel (four interleaved running sums).
__device__ __forceinline__ double sum_slices(const rpy::PartialSums& ps, int64_t e)
{
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int c = 0;
    for (; c + 4 <= ps.n_slices; c += 4) {
        s0 += ps.partial[(int64_t)c * ps.per_chunk + e];
        s1 += ps.partial[(int64_t)(c + 1) * ps.per_chunk + e];
        s2 += ps.partial[(int64_t)(c + 2) * ps.per_chunk + e];
        s3 += ps.partial[(int64_t)(c + 3) * ps.per_chunk + e];
    }
    for (; c < ps.n_slices; ++c) s0 += ps.partial[(int64_t)c * ps.per_chunk + e];
    return ((s0 + s1) + (s2 + s3)) * ps.scale;
}

// The two O(N) pieces of Eq. (11)'s operator in one pass, one warp per body (blockIdx.y = right-hand side):
//   out_top[i]  = (M lambda)_i - (K U)_i
//   out_bot[p]  = -(K^T lambda)_p
// in = [lambda; U], out = [top; bottom], both with `stride` doubles between right-hand sides.  M lambda comes
// from the product's per-slice partial sums when ps.partial is set (the product's finalise step fused in here:
// one launch less per iteration, and the fp32 path's result is not rounded to float on the way), else from
// vel32 (float), else it is already in out_top.
__global__ void saddle_tail_kernel(const double* __restrict__ pos, const double* __restrict__ q,
                                   const int64_t* __restrict__ offsets, const double* __restrict__ in,
                                   const float* __restrict__ vel32, double* __restrict__ out,
                                   int64_t n_blobs, int64_t n_bodies, int64_t stride, rpy::PartialSums ps,
                                   const int* __restrict__ skip)
{
    rpy::pdl_enter();
    const int64_t p = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (skip != nullptr && *skip != 0) return;
    in += (int64_t)blockIdx.y * stride; out += (int64_t)blockIdx.y * stride;
    if (vel32) vel32 += (int64_t)blockIdx.y * 3 * n_blobs;
    if (ps.partial) {
        // the bodies of this CTA own a contiguous range of output elements: all threads add the slices for it
        // (one element per thread and pass, coalesced in every slice), then each warp goes on with its body
        const int64_t pA = (int64_t)blockIdx.x * (blockDim.x >> 5);
        const int64_t pB = pA + (blockDim.x >> 5) < n_bodies ? pA + (blockDim.x >> 5) : n_bodies;
        if (pA < n_bodies) {
            const int64_t e1 = 3 * offsets[pB], base = (int64_t)blockIdx.y * n_blobs * 3;
            for (int64_t e = 3 * offsets[pA] + threadIdx.x; e < e1; e += blockDim.x) out[e] = sum_slices(ps, base + e);
        }
        __syncthreads();
    }
    if (p >= n_bodies) return;
    const double* U = in + 3 * n_blobs + 6 * p;
    const double ux = U[0], uy = U[1], uz = U[2], wx = U[3], wy = U[4], wz = U[5];
    const double qx = q[3 * p + 0], qy = q[3 * p + 1], qz = q[3 * p + 2];
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int64_t i = offsets[p] + lane; i < offsets[p + 1]; i += 32) {
        const double dx = pos[3 * i + 0] - qx, dy = pos[3 * i + 1] - qy, dz = pos[3 * i + 2] - qz;
        double m0, m1, m2;
        if (vel32) {
            m0 = (double)vel32[3 * i + 0]; m1 = (double)vel32[3 * i + 1]; m2 = (double)vel32[3 * i + 2];
        } else {
            m0 = out[3 * i + 0]; m1 = out[3 * i + 1]; m2 = out[3 * i + 2];
        }
        out[3 * i + 0] = m0 - (ux + (wy * dz - wz * dy));
        out[3 * i + 1] = m1 - (uy + (wz * dx - wx * dz));
        out[3 * i + 2] = m2 - (uz + (wx * dy - wy * dx));
        const double lx = in[3 * i + 0], ly = in[3 * i + 1], lz = in[3 * i + 2];
        s[0] += lx; s[1] += ly; s[2] += lz;
        s[3] += dy * lz - dz * ly;
        s[4] += dz * lx - dx * lz;
        s[5] += dx * ly - dy * lx;
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) s[c] = warp_sum(s[c]);
    if (lane < 6) {
        double v = s[0];
#pragma unroll
        for (int c = 1; c < 6; ++c) if (lane == c) v = s[c];
        out[3 * n_blobs + 6 * p + lane] = -v;
    }
}

// r = c_p + R(theta_p) t, R from the unit quaternion (s, p): the standard rotation matrix.
template <class S>
__global__ void blob_positions_kernel(const S* __restrict__ tmpl, const S* __restrict__ centres,
                                      const S* __restrict__ quats, S* __restrict__ pos, int64_t n_bodies, int bpb)
{
    const int64_t total = n_bodies * bpb;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t p = e / bpb;
        const int t = (int)(e % bpb);
        double s = quats[4 * p + 0], x = quats[4 * p + 1], y = quats[4 * p + 2], z = quats[4 * p + 3];
        const double nrm = 1.0 / sqrt(s * s + x * x + y * y + z * z);
        s *= nrm; x *= nrm; y *= nrm; z *= nrm;
        const double tx = tmpl[3 * t + 0], ty = tmpl[3 * t + 1], tz = tmpl[3 * t + 2];
        const double rx = (1 - 2 * (y * y + z * z)) * tx + 2 * (x * y - s * z) * ty + 2 * (x * z + s * y) * tz;
        const double ry = 2 * (x * y + s * z) * tx + (1 - 2 * (x * x + z * z)) * ty + 2 * (y * z - s * x) * tz;
        const double rz = 2 * (x * z - s * y) * tx + 2 * (y * z + s * x) * ty + (1 - 2 * (x * x + y * y)) * tz;
        pos[3 * e + 0] = (S)((double)centres[3 * p + 0] + rx);
        pos[3 * e + 1] = (S)((double)centres[3 * p + 1] + ry);
        pos[3 * e + 2] = (S)((double)centres[3 * p + 2] + rz);
    }
}

// ------------------------------------------------------------------ preconditioner storage
// [header 4 x int64][offsets nb+1][mat_off nb+1][info nb x int32][factors][Y 3N x 6][Nt nb x 36]
struct PrecondLayout {
    size_t offsets_at, matoff_at, info_at, factors_at, y_at, nt_at, total;
    int64_t n_blobs, total_mat;
    int max_m;
};

bool layout_of(int64_t nb, const int64_t* h_off, PrecondLayout& L)
{
    if (nb < 1 || !h_off || h_off[0] != 0) return false;
    int64_t tot = 0; int max_m = 0;
    for (int64_t p = 0; p < nb; ++p) {
        int64_t c = h_off[p + 1] - h_off[p];
        if (c < 1 || c > RPY_RIGID_MAX_BODY_BLOBS) return false;
        tot += 9 * c * c;
        if (3 * c > max_m) max_m = (int)(3 * c);
    }
    L.n_blobs = h_off[nb]; L.total_mat = tot; L.max_m = max_m;
    size_t at = align_up(4 * sizeof(int64_t), kAlign);
    L.offsets_at = at; at = align_up(at + (size_t)(nb + 1) * 8, kAlign);
    L.matoff_at = at;  at = align_up(at + (size_t)(nb + 1) * 8, kAlign);
    L.info_at = at;    at = align_up(at + (size_t)nb * 4, kAlign);
    L.factors_at = at; at = align_up(at + (size_t)tot * 8, kAlign);
    L.y_at = at;       at = align_up(at + (size_t)L.n_blobs * 18 * 8, kAlign);
    L.nt_at = at;      at = align_up(at + (size_t)nb * 36 * 8, kAlign);
    L.total = at;
    return true;
}

// Device-side view rebuilt from (n_blobs, n_bodies, total_mat) without the host offsets.
struct PrecondView {
    const int64_t* offsets; const int64_t* mat_off; int* info; double* factors; double* Y; double* Nt;
};
__host__ __device__ inline size_t align_up_hd(size_t x) { return (x + 255) / 256 * 256; }
// header: [0] magic, [1] n_bodies, [2] n_blobs, [3] total_mat (doubles in the factor region),
//         [4] first body whose factorisation failed, -1 if none (written by precond_finish_kernel)
constexpr int kHdrWords = 5;
__host__ __device__ inline PrecondView view_of(void* base, int64_t nb, int64_t n_blobs, int64_t total_mat)
{
    unsigned char* b = static_cast<unsigned char*>(base);
    size_t at = align_up_hd(4 * sizeof(int64_t));
    PrecondView v;
    v.offsets = reinterpret_cast<const int64_t*>(b + at); at = align_up_hd(at + (size_t)(nb + 1) * 8);
    v.mat_off = reinterpret_cast<const int64_t*>(b + at); at = align_up_hd(at + (size_t)(nb + 1) * 8);
    v.info = reinterpret_cast<int*>(b + at);              at = align_up_hd(at + (size_t)nb * 4);
    v.factors = reinterpret_cast<double*>(b + at);        at = align_up_hd(at + (size_t)total_mat * 8);
    v.Y = reinterpret_cast<double*>(b + at);              at = align_up_hd(at + (size_t)n_blobs * 18 * 8);
    v.Nt = reinterpret_cast<double*>(b + at);
    return v;
}

// ------------------------------------------------------------------ dense 3x3 block (double lanes)
// The block M_ij * (6 pi eta a) from the matvec's own pair arithmetic: the five collected scalars of
// rpy_math.cuh give  [al + be dx dx, be dx dy, ga dx; be dx dy, al + be dy dy, ga dy; ep dx, ep dy, de]
// (wall) or f I + G d d^T (free).  Positions are already divided by a.
template <bool WALL>
__device__ __forceinline__ void pair_block(double xi, double yi, double zi, double xj, double yj, double zj,
                                           double B[9])
{
    using L = rpy::Lane<double>;
    rpy::PairCoef<double> c;
    rpy::PairPre<double> pre;
    rpy::pair_pre<L, WALL>(xi, yi, zi, xj, yj, zj, c, pre);
    if (pre.r2 <= 4.0) rpy::rpy_near_fixup<L, WALL>(pre.r2, pre.n1, pre.f, pre.G);
    rpy::pair_post<L, WALL>(2.0 * zi, zj, pre, c);
    const double f = pre.f, G = pre.G;
    if (WALL) {
        B[0] = c.al + c.be * c.dx * c.dx; B[1] = c.be * c.dx * c.dy;        B[2] = c.ga * c.dx;
        B[3] = B[1];                      B[4] = c.al + c.be * c.dy * c.dy; B[5] = c.ga * c.dy;
        B[6] = c.ep * c.dx;               B[7] = c.ep * c.dy;               B[8] = c.de;
    } else {
        B[0] = f + G * c.dx * c.dx; B[1] = G * c.dx * c.dy;     B[2] = G * c.dx * c.dz;
        B[3] = B[1];                B[4] = f + G * c.dy * c.dy; B[5] = G * c.dy * c.dz;
        B[6] = B[2];                B[7] = B[5];                B[8] = f + G * c.dz * c.dz;
    }
}

// Pseudo-inverse of the symmetric positive SEMI-definite 6x6 K_p^T (M^(pp))^-1 K_p ("in practice all
// inverses should be replaced by pseudo-inverses"): cyclic Jacobi eigen-decomposition,
// eigenvalues below 1e-10 of the largest are dropped (a straight line of blobs cannot resist a torque
// about its axis: that direction gets zero mobility), a negative or non-finite spectrum fails.
__device__ bool sym6_pinv(const double* __restrict__ a_in, double* __restrict__ out)
{
    // every index below is a compile-time constant after unrolling: both matrices live in registers
    double a[6][6], v[6][6];
#pragma unroll
    for (int r = 0; r < 6; ++r)
#pragma unroll
        for (int c = 0; c < 6; ++c) { a[r][c] = 0.5 * (a_in[6 * r + c] + a_in[6 * c + r]); v[r][c] = r == c ? 1.0 : 0.0; }
#pragma unroll 1
    for (int sweep = 0; sweep < 30; ++sweep) {
        double off = 0.0, diag = 0.0;
#pragma unroll
        for (int r = 0; r < 6; ++r)
#pragma unroll
            for (int c = 0; c < 6; ++c) { if (r != c) off += a[r][c] * a[r][c]; else diag += a[r][c] * a[r][c]; }
        if (!(off > 1e-60 * diag) || !isfinite(off)) break;
#pragma unroll
        for (int p = 0; p < 5; ++p)
#pragma unroll
            for (int q = p + 1; q < 6; ++q) {
                if (a[p][q] != 0.0) {
                    const double theta = (a[q][q] - a[p][p]) / (2.0 * a[p][q]);
                    const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                    const double c = rsqrt(t * t + 1.0), sn = t * c;
                    const double app = a[p][p], aqq = a[q][q], apq = a[p][q];
#pragma unroll
                    for (int k = 0; k < 6; ++k) {              // rows / columns p and q of J^T A J, k != p, q
                        if (k != p && k != q) {
                            const double akp = a[k][p], akq = a[k][q];
                            a[k][p] = a[p][k] = c * akp - sn * akq;
                            a[k][q] = a[q][k] = sn * akp + c * akq;
                        }
                    }
                    a[p][p] = c * c * app - 2.0 * c * sn * apq + sn * sn * aqq;
                    a[q][q] = sn * sn * app + 2.0 * c * sn * apq + c * c * aqq;
                    a[p][q] = a[q][p] = 0.0;
#pragma unroll
                    for (int k = 0; k < 6; ++k) {              // V <- V J
                        const double vkp = v[k][p], vkq = v[k][q];
                        v[k][p] = c * vkp - sn * vkq; v[k][q] = sn * vkp + c * vkq;
                    }
                }
            }
    }
    double lmax = 0.0;
    bool finite = true;
#pragma unroll
    for (int i = 0; i < 6; ++i) { finite = finite && isfinite(a[i][i]); if (a[i][i] > lmax) lmax = a[i][i]; }
    if (!finite || !(lmax > 0.0)) return false;
    double inv[6];
    bool negative = false;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        negative = negative || a[i][i] < -1e-10 * lmax;
        inv[i] = a[i][i] > 1e-10 * lmax ? 1.0 / a[i][i] : 0.0;
    }
    if (negative) return false;
#pragma unroll
    for (int r = 0; r < 6; ++r)
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            double sum = 0.0;
#pragma unroll
            for (int i = 0; i < 6; ++i) sum += v[r][i] * v[c][i] * inv[i];
            out[6 * r + c] = sum;
        }
    return true;
}

// ------------------------------------------------------------------ preconditioner build
// One CTA per body.  A (m x m, leading dimension ld) is in shared memory when m <= kSmemBodyM, else
// it is the body's slot of `factors` (ld = m).  Steps: fill M^(pp); right-looking Cholesky on the
// lower triangle, one barrier per column (the 256 threads tile the trailing triangle 16 x 16:
// thread (tx, ty) updates A[i][k] for i = j+1+ty+16a, k = j+1+tx+16b <= i; a half-warp touches 16
// consecutive doubles of one row); the inverse (M^(pp))^-1 = L^-T L^-1 formed in place from the factor;
// Y = (M^(pp))^-1 K_p; N~ = (K_p^T Y)^-1 by Gauss-Jordan on the 6x6; store the full symmetric inverse.
template <bool WALL>
__global__ void __launch_bounds__(kBuildThreads)
precond_build_kernel(const double* __restrict__ pos, const double* __restrict__ q,
                     const int64_t* __restrict__ offsets, const int64_t* __restrict__ mat_off,
                     int* __restrict__ info, double* __restrict__ factors, double* __restrict__ Yg,
                     double* __restrict__ Ntg, double inv_a, double scale, int only_above)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ double s_n[36];
    __shared__ int s_fail;
    const int p = blockIdx.x, tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const int64_t b0 = offsets[p];
    const int nbp = (int)(offsets[p + 1] - b0);
    const int m = 3 * nbp;
    if (m <= only_above) return;                               // precond_build_reg_kernel takes this body
    const bool in_smem = m <= kSmemBodyM;
    double* const G = factors + mat_off[p];
    const int ld = in_smem ? (m | 1) : m;
    double* const A = in_smem ? sm : G;
    double* const Yb = in_smem ? sm + (size_t)ld * m : Yg + b0 * 18;      // [m][6]
    if (tid == 0) s_fail = 0;

    for (int e = tid; e < nbp * nbp; e += kBuildThreads) {
        const int bi = e / nbp, bj = e % nbp;
        const double* ri = pos + 3 * (b0 + bi);
        const double* rj = pos + 3 * (b0 + bj);
        double B[9];
        pair_block<WALL>(ri[0] * inv_a, ri[1] * inv_a, ri[2] * inv_a, rj[0] * inv_a, rj[1] * inv_a, rj[2] * inv_a, B);
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) A[(size_t)(3 * bi + r) * ld + 3 * bj + c] = scale * B[3 * r + c];
    }
    __syncthreads();

    for (int j = 0; j < m; ++j) {
        const double d = A[(size_t)j * ld + j];
        if (!(d > 0.0) || !isfinite(d)) { if (tid == 0) s_fail = j + 1; break; }   // uniform: all threads read the same d
        const double rd = 1.0 / d;
        // trailing update A[i][k] -= A[i][j] A[k][j] / d for j < k <= i: 16 x 16 thread tile over (i, k)
        for (int i = j + 1 + ty; i < m; i += 16) {
            const double lij = A[(size_t)i * ld + j] * rd;
            double* Ai = A + (size_t)i * ld;
            int k = j + 1 + tx;
            for (; k + 48 <= i; k += 64) {           // four independent load-FMA-store chains in flight
                const double c0 = A[(size_t)k * ld + j], c1 = A[(size_t)(k + 16) * ld + j];
                const double c2 = A[(size_t)(k + 32) * ld + j], c3 = A[(size_t)(k + 48) * ld + j];
                const double a0 = Ai[k], a1 = Ai[k + 16], a2 = Ai[k + 32], a3 = Ai[k + 48];
                Ai[k] = a0 - lij * c0; Ai[k + 16] = a1 - lij * c1;
                Ai[k + 32] = a2 - lij * c2; Ai[k + 48] = a3 - lij * c3;
            }
            for (; k <= i; k += 16) Ai[k] -= lij * A[(size_t)k * ld + j];
        }
        __syncthreads();
        const double rs = 1.0 / sqrt(d);
        for (int i = j + tid; i < m; i += kBuildThreads)
            A[(size_t)i * ld + j] = i == j ? sqrt(d) : A[(size_t)i * ld + j] * rs;
    }
    __syncthreads();
    if (s_fail) {
        if (tid == 0) info[p] = s_fail;
        return;
    }

    // ---- explicit inverse ("dense matrix inversion (e.g., Cholesky factorization)"):
    // Z = L^-1 in place (column by column from the right: Z[j+1:, j] = -Z[j+1:, j+1:] L[j+1:, j] / L_jj,
    // thread i takes row i of the product, the column is first copied to `tmp`), then
    // M^-1 = Z^T Z in place on the lower triangle (row i from rows k >= i, thread c takes column c).
    double* const tmp = Yb;
    for (int j = m - 1; j >= 0; --j) {
        const double ajj = 1.0 / A[(size_t)j * ld + j];
        for (int i = j + 1 + tid; i < m; i += kBuildThreads) tmp[i] = A[(size_t)i * ld + j];
        __syncthreads();
        for (int i = j + 1 + tid; i < m; i += kBuildThreads) {
            const double* Ai = A + (size_t)i * ld;
            double sum = 0.0;
            for (int k = j + 1; k <= i; ++k) sum += Ai[k] * tmp[k];
            A[(size_t)i * ld + j] = -ajj * sum;
        }
        if (tid == 0) A[(size_t)j * ld + j] = ajj;
        __syncthreads();
    }
    for (int i = 0; i < m; ++i) {
        for (int c0 = 0; c0 <= i; c0 += kBuildThreads) {    // chunks of columns; column i itself is in the last one
            const int c = c0 + tid;
            double sum = 0.0;
            if (c <= i)
                for (int k = i; k < m; ++k) sum += A[(size_t)k * ld + i] * A[(size_t)k * ld + c];
            __syncthreads();                               // every thread has read row i and column i
            if (c <= i) A[(size_t)i * ld + c] = sum;
            __syncthreads();
        }
    }
    // mirror: A[c][i] = A[i][c] so that rows are complete
    for (int e = tid; e < m * m; e += kBuildThreads) {
        const int i = e / m, c = e % m;
        if (c > i) A[(size_t)i * ld + c] = A[(size_t)c * ld + i];
    }
    __syncthreads();

    // Y = M^-1 K_p.  K_p rows of blob b (real lengths): [I | C_b], C_b = [[0, dz, -dy], [-dz, 0, dx], [dy, -dx, 0]]
    const double qx = q[3 * p + 0], qy = q[3 * p + 1], qz = q[3 * p + 2];
    for (int e = tid; e < m * 6; e += kBuildThreads) {
        const int i = e / 6, c = e % 6;
        const double* Ai = A + (size_t)i * ld;
        double sum = 0.0;
        if (c < 3) {
            for (int bb = 0; bb < nbp; ++bb) sum += Ai[3 * bb + c];
        } else {
            for (int bb = 0; bb < nbp; ++bb) {
                const double* rb = pos + 3 * (b0 + bb);
                const double dx = rb[0] - qx, dy = rb[1] - qy, dz = rb[2] - qz;
                const double m0 = Ai[3 * bb], m1 = Ai[3 * bb + 1], m2 = Ai[3 * bb + 2];
                sum += c == 3 ? (m2 * dy - m1 * dz) : c == 4 ? (m0 * dz - m2 * dx) : (m1 * dx - m0 * dy);
            }
        }
        Yg[b0 * 18 + e] = sum;
    }
    __syncthreads();
    if (tid < 36) {                                          // K_p^T Y
        const int r = tid / 6, c = tid % 6;
        const double* Y = Yg + b0 * 18;
        double sum = 0.0;
        for (int bb = 0; bb < nbp; ++bb) {
            const double y0 = Y[(size_t)(3 * bb) * 6 + c], y1 = Y[(size_t)(3 * bb + 1) * 6 + c], y2 = Y[(size_t)(3 * bb + 2) * 6 + c];
            if (r < 3) sum += r == 0 ? y0 : r == 1 ? y1 : y2;
            else {
                const double* rb = pos + 3 * (b0 + bb);
                const double dx = rb[0] - qx, dy = rb[1] - qy, dz = rb[2] - qz;
                sum += r == 3 ? (dy * y2 - dz * y1) : r == 4 ? (dz * y0 - dx * y2) : (dx * y1 - dy * y0);
            }
        }
        s_n[tid] = sum;
    }
    __syncthreads();
    if (tid == 0) {
        // The 6x6 mixes a force/velocity block (~ eta L), two coupling blocks (~ eta L^2) and a torque/angular
        // velocity block (~ eta L^3): its spectrum, and with it the cut-off of the pseudo-inverse, would depend
        // on the unit of length.  Lengths are therefore taken in units of the blob radius first, S' = D S D with
        // D = diag(1, 1, 1, 1/a, 1/a, 1/a), and the result is scaled back, S^+ := D S'^+ D (reading A18).
        double sc[36], nt[36];
        for (int e = 0; e < 36; ++e) sc[e] = s_n[e] * (e / 6 >= 3 ? inv_a : 1.0) * (e % 6 >= 3 ? inv_a : 1.0);
        const bool ok = sym6_pinv(sc, nt);
        for (int e = 0; e < 36; ++e)
            Ntg[(size_t)p * 36 + e] = ok ? nt[e] * (e / 6 >= 3 ? inv_a : 1.0) * (e % 6 >= 3 ? inv_a : 1.0) : 0.0;
        info[p] = ok ? 0 : m + 1;
    }
    if (in_smem)
        for (int e = tid; e < m * m; e += kBuildThreads) G[e] = A[(size_t)(e / m) * ld + e % m];
}

// ------------------------------------------------------------------ preconditioner build, register-resident
// Bodies with m = 3 n_p <= kRegMaxM (the paper's: 12-42 blobs per body): the matrix never
// sits in shared memory.  The augmented symmetric matrix
//     A = [ M^(pp)   K_p ]        (m padded to a multiple of 8 with an identity block; K_p padded to 8 columns)
//         [ K_p^T    0   ]
// is cut into 8 x 8 tiles of its lower triangle, ONE TILE PER THREAD, held in 64 double registers for the
// whole kernel.  The block form of the symmetric sweep operator is applied to the pivot blocks p of M^(pp)
// (4 rows each) in turn:
//     P = A_pp^-1,  W = A_{:,p} P,   A <- A - W A_{:,p}^T  everywhere,   then  A_{:,p} = W,  A_pp = -P,
// the same formula for blocks already swept and blocks still to come, so every thread does the same work
// in every step and nothing shrinks.  After all pivot blocks of M^(pp):
//     A = [ -(M^(pp))^-1           (M^(pp))^-1 K_p      ]     i.e. the explicit inverse ("dense matrix
//         [ K_p^T (M^(pp))^-1     -K_p^T (M^(pp))^-1 K_p ]     inversion"), Y and the 6 x 6
// Schur complement of Eq. (19) in one pass, m^3/2 fused multiply-adds, the work of Cholesky
// + triangular inverse + L^-T L^-1.  A step exchanges only the m x 4 panel A_{:,p} and W through shared
// memory (two barriers, panels double-buffered): each thread loads 2 x 8 doubles per 64 multiply-adds.
// The pivots of the 4 x 4 blocks are Schur complements of an SPD matrix: a non-positive one reports the body
// as not positive definite, as the Cholesky factorisation did.
constexpr int kRT = 8;                         // thread tile
constexpr int kRegMaxM = 128;                  // largest m = 3 n_p on this path
constexpr int kRegMaxTA = kRegMaxM / kRT + 1;  // tile rows incl. the K^T row
constexpr int kRegMaxThreads = 160;            // >= 17 * 18 / 2 = 153 tiles
constexpr int kPanelStride = 10;               // doubles per 8 panel rows in shared memory (spreads the banks)
constexpr int kPanelLen = kRegMaxTA * kPanelStride;

__device__ __forceinline__ int panel_at(int row) { return (row >> 3) * kPanelStride + (row & 7); }

// K_p[3 b + comp][c] for the blob at d = r_b - q_p: [I | C_b], C_b = [[0, dz, -dy], [-dz, 0, dx], [dy, -dx, 0]]
__device__ __forceinline__ double k_entry(int comp, int c, double dx, double dy, double dz)
{
    if (c < 3) return comp == c ? 1.0 : 0.0;
    const int cc = c - 3;
    if (comp == cc) return 0.0;
    if (comp == 0) return cc == 1 ? dz : -dy;
    if (comp == 1) return cc == 0 ? -dz : dx;
    return cc == 0 ? dy : -dx;
}

// P = B^-1 for the symmetric positive definite 4 x 4 block B = A[PO..PO+3][PO..PO+3] of a diagonal tile, by four
// scalar sweeps (all indices compile-time).  Returns false when a pivot is not positive and finite.
template <int PO>
__device__ __forceinline__ bool pivot_inverse(const double (&A)[kRT][kRT], double (&P)[4][4])
{
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) P[i][j] = A[PO + i][PO + j];
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double d = P[k][k];
        ok = ok && d > 0.0 && isfinite(d);
        // 1/d for a positive finite pivot: the MUFU.RCP64H seed and two Newton steps.  The four pivots of a block are
        // inverted one after the other by ONE thread while the CTA waits, so the division's slow path was on the critical
        // path (cfg 3 build 1.88 -> 1.75 ms; the inverse unchanged to 13 digits)
        double inv;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(inv) : "d"(d));
        inv = fma(inv, fma(-d, inv, 1.0), inv);
        inv = fma(inv, fma(-d, inv, 1.0), inv);
        double w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) w[i] = P[i][k] * inv;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (i != k && j != k) P[i][j] = fma(-w[i], P[k][j], P[i][j]);
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (i != k) { P[i][k] = w[i]; P[k][i] = w[i]; }
        P[k][k] = -inv;
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) P[i][j] = -P[i][j];       // the sweeps leave -B^-1
    return ok;
}

// One sweep step for pivot rows 8 Pt + PO .. + 3 (PO = 0 or 4, compile-time so that the register tile is only
// ever indexed with constants).  Cp, Wp: this step's panel buffers [4][kPanelLen]; Pm: its 4 x 4 inverse.
template <int PO>
__device__ __forceinline__ void sweep_step(double (&A)[kRT][kRT], bool has_tile, int I, int J, int Pt, int n_rows,
                                           double* __restrict__ Cp, double* __restrict__ Wp, double* __restrict__ Pm,
                                           int* s_fail, int step_no)
{
    // (a) the panel A_{:,p}: rows of tile row I from the tiles (I, Pt), I >= Pt; rows of tile row J < Pt from the
    //     transposes of the tiles (Pt, J); the owner of (Pt, Pt) also inverts the pivot block
    if (has_tile && J == Pt) {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int r = 0; r < kRT; ++r) Cp[c * kPanelLen + I * kPanelStride + r] = A[r][PO + c];
        if (I == Pt) {
            double P[4][4];
            if (!pivot_inverse<PO>(A, P)) *s_fail = step_no + 1;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) Pm[4 * i + j] = P[i][j];
        }
    } else if (has_tile && I == Pt) {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int q = 0; q < kRT; ++q) Cp[c * kPanelLen + J * kPanelStride + q] = A[PO + c][q];
    }
    __syncthreads();
    if (*s_fail) return;                                      // uniform: written before the barrier
    // (b) W = A_{:,p} P, one row per thread
    for (int i = threadIdx.x; i < n_rows; i += blockDim.x) {
        const int at = panel_at(i);
        const double c0 = Cp[at], c1 = Cp[kPanelLen + at], c2 = Cp[2 * kPanelLen + at], c3 = Cp[3 * kPanelLen + at];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            Wp[j * kPanelLen + at] = fma(c3, Pm[12 + j], fma(c2, Pm[8 + j], fma(c1, Pm[4 + j], c0 * Pm[j])));
    }
    __syncthreads();
    if (!has_tile) return;
    // (c) A_IJ -= W_I A_{J,p}^T
#pragma unroll 1
    for (int c = 0; c < 4; ++c) {
        double w[kRT], cj[kRT];
        const double2* wp = reinterpret_cast<const double2*>(Wp + c * kPanelLen + I * kPanelStride);
        const double2* cp = reinterpret_cast<const double2*>(Cp + c * kPanelLen + J * kPanelStride);
#pragma unroll
        for (int h = 0; h < kRT / 2; ++h) {
            const double2 a = wp[h], b = cp[h];
            w[2 * h] = a.x; w[2 * h + 1] = a.y; cj[2 * h] = b.x; cj[2 * h + 1] = b.y;
        }
#pragma unroll
        for (int r = 0; r < kRT; ++r)
#pragma unroll
            for (int q = 0; q < kRT; ++q) A[r][q] = fma(-w[r], cj[q], A[r][q]);
    }
    // (d) the pivot rows and columns themselves: A_{:,p} = W, A_{p,:} = W^T, A_pp = -P
    if (J == Pt) {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int r = 0; r < kRT; ++r) A[r][PO + c] = Wp[c * kPanelLen + I * kPanelStride + r];
    }
    if (I == Pt) {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int q = 0; q < kRT; ++q) A[PO + c][q] = Wp[c * kPanelLen + J * kPanelStride + q];
        if (J == Pt) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) A[PO + i][PO + j] = -Pm[4 * i + j];
        }
    }
}

template <bool WALL>
// Two CTAs per SM need <= 168 registers: each SM sub-partition holds 16,384 and gets three of the ten warps.
__global__ void __launch_bounds__(kRegMaxThreads, 2)
precond_build_reg_kernel(const double* __restrict__ pos, const double* __restrict__ q,
                         const int64_t* __restrict__ offsets, const int64_t* __restrict__ mat_off,
                         int* __restrict__ info, double* __restrict__ factors, double* __restrict__ Yg,
                         double* __restrict__ Ntg, double inv_a, double scale)
{
    __shared__ __align__(16) double s_C[2][4 * kPanelLen];
    __shared__ __align__(16) double s_W[2][4 * kPanelLen];
    __shared__ __align__(16) double s_P[2][16];
    __shared__ int s_fail;
    const int p = blockIdx.x, tid = threadIdx.x;
    const int64_t b0 = offsets[p];
    const int nbp = (int)(offsets[p + 1] - b0);
    const int m = 3 * nbp;
    if (m > kRegMaxM) return;                                  // the shared/global-memory kernel takes this body
    double* const G = factors + mat_off[p];
    const int T = (m + kRT - 1) / kRT, TA = T + 1;             // tile rows of M^(pp); with the K^T row
    const int n_tiles = TA * (TA + 1) / 2;
    if (tid == 0) s_fail = 0;

    // M^(pp) into the body's slot of `factors` (overwritten by the inverse at the end): one pair block per
    // unordered blob pair, written with its transpose (M_ji = M_ij^T)
    for (int e = tid; e < nbp * (nbp + 1) / 2; e += blockDim.x) {
        int bi = (int)((sqrtf(8.0f * (float)e + 1.0f) - 1.0f) * 0.5f);
        while ((bi + 1) * (bi + 2) / 2 <= e) ++bi;
        while (bi * (bi + 1) / 2 > e) --bi;
        const int bj = e - bi * (bi + 1) / 2;
        const double* ri = pos + 3 * (b0 + bi);
        const double* rj = pos + 3 * (b0 + bj);
        double B[9];
        pair_block<WALL>(ri[0] * inv_a, ri[1] * inv_a, ri[2] * inv_a, rj[0] * inv_a, rj[1] * inv_a, rj[2] * inv_a, B);
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                G[(size_t)(3 * bi + r) * m + 3 * bj + c] = scale * B[3 * r + c];
                G[(size_t)(3 * bj + c) * m + 3 * bi + r] = scale * B[3 * r + c];
            }
    }
    __syncthreads();

    // this thread's tile (I, J), J <= I, of the augmented matrix
    const bool has_tile = tid < n_tiles;
    int I = 0;
    while ((I + 1) * (I + 2) / 2 <= tid) ++I;
    const int J = tid - I * (I + 1) / 2;
    const double qx = q[3 * p + 0], qy = q[3 * p + 1], qz = q[3 * p + 2];
    double A[kRT][kRT];
    if (has_tile) {
#pragma unroll
        for (int r = 0; r < kRT; ++r)
#pragma unroll
            for (int c = 0; c < kRT; ++c) {
                const int gi = kRT * I + r, gj = kRT * J + c;
                double v;
                if (I < T) v = (gi < m && gj < m) ? G[(size_t)gi * m + gj] : (gi == gj ? 1.0 : 0.0);
                else if (J < T && r < 6 && gj < m) {              // row r of K_p^T
                    const double* rb = pos + 3 * (b0 + gj / 3);
                    v = k_entry(gj % 3, r, rb[0] - qx, rb[1] - qy, rb[2] - qz);
                } else v = 0.0;
                A[r][c] = v;
            }
    }
    __syncthreads();                                           // everyone has read M^(pp) from G

    const int n_rows = kRT * TA;
    for (int s = 0; s < 2 * T; ++s) {
        const int b = s & 1;
        if (s & 1) sweep_step<4>(A, has_tile, I, J, s >> 1, n_rows, s_C[b], s_W[b], s_P[b], &s_fail, s);
        else       sweep_step<0>(A, has_tile, I, J, s >> 1, n_rows, s_C[b], s_W[b], s_P[b], &s_fail, s);
        if (s_fail) break;                                     // uniform (see sweep_step)
    }
    if (s_fail) {
        if (tid == 0) info[p] = s_fail;
        return;
    }
    if (tid == 0) info[p] = 0;
    if (!has_tile) return;
    if (I < T) {                                               // (M^(pp))^-1, full symmetric storage
#pragma unroll
        for (int r = 0; r < kRT; ++r)
#pragma unroll
            for (int c = 0; c < kRT; ++c) {
                const int gi = kRT * I + r, gj = kRT * J + c;
                if (gi < m && gj < m && (I != J || c <= r)) {      // a diagonal tile stores its lower half twice:
                    G[(size_t)gi * m + gj] = -A[r][c];             // the result is symmetric bit for bit
                    G[(size_t)gj * m + gi] = -A[r][c];
                }
            }
    } else if (J < T) {                                        // Y = (M^(pp))^-1 K_p, [m][6]
#pragma unroll
        for (int r = 0; r < 6; ++r)
#pragma unroll
            for (int c = 0; c < kRT; ++c) {
                const int gj = kRT * J + c;
                if (gj < m) Yg[b0 * 18 + (size_t)gj * 6 + r] = A[r][c];
            }
    } else {                                                   // K_p^T (M^(pp))^-1 K_p, inverted by ntilde_kernel
#pragma unroll
        for (int r = 0; r < 6; ++r)
#pragma unroll
            for (int c = 0; c < 6; ++c) Ntg[(size_t)p * 36 + 6 * r + c] = -A[r][c];
    }
}

// N~_pp = (K_p^T (M^(pp))^-1 K_p)^+ in place for the bodies of the register path, one thread per body.
// The 6x6 mixes a force/velocity block (~ eta L), two coupling blocks (~ eta L^2) and a torque/angular velocity
// block (~ eta L^3): its spectrum, and with it the cut-off of the pseudo-inverse, would depend on the unit of
// length.  Lengths are therefore taken in units of the blob radius first, S' = D S D with
// D = diag(1, 1, 1, 1/a, 1/a, 1/a), and the result is scaled back, S^+ := D S'^+ D (reading A18).
__global__ void ntilde_kernel(const int64_t* __restrict__ offsets, int* __restrict__ info, double* __restrict__ Ntg,
                              int64_t n_bodies, double inv_a)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_bodies) return;
    const int m = 3 * (int)(offsets[p + 1] - offsets[p]);
    if (m > kRegMaxM || info[p] != 0) return;
    double sc[36], nt[36];
    for (int e = 0; e < 36; ++e) sc[e] = Ntg[p * 36 + e] * (e / 6 >= 3 ? inv_a : 1.0) * (e % 6 >= 3 ? inv_a : 1.0);
    const bool ok = sym6_pinv(sc, nt);
    for (int e = 0; e < 36; ++e)
        Ntg[p * 36 + e] = ok ? nt[e] * (e / 6 >= 3 ? inv_a : 1.0) * (e % 6 >= 3 ? inv_a : 1.0) : 0.0;
    if (!ok) info[p] = m + 1;
}

// After the build: header word 4 = the first body whose info is non-zero (-1: none), so that reading the
// outcome later is a read-only copy of the header.  One CTA.
__global__ void precond_finish_kernel(const int* __restrict__ info, int64_t n_bodies, int64_t* __restrict__ hdr)
{
    __shared__ long long s_min;
    if (threadIdx.x == 0) s_min = (long long)1 << 62;
    __syncthreads();
    long long mine = (long long)1 << 62;
    for (int64_t p = threadIdx.x; p < n_bodies; p += blockDim.x)
        if (info[p] != 0 && p < mine) mine = p;
    if (mine != ((long long)1 << 62)) atomicMin(&s_min, mine);
    __syncthreads();
    if (threadIdx.x == 0) hdr[4] = s_min == ((long long)1 << 62) ? -1 : s_min;
}

// ------------------------------------------------------------------ preconditioner apply
// [lambda; U] = P_p^-1 [x; y] (Eq. (19)):
//   r = Y^T x (= K^T M^-1 x),  U = -N~ (y + r),  t = M^-1 x,  lambda = t + Y U.
// t = (M^(pp))^-1 x is a dense symmetric matrix-vector product: lane l owns rows l, l+32, ... in chunks of 128
// rows and walks the columns j, reading the contiguous row j of the stored inverse (= its column j) --
// coalesced, every load independent of the arithmetic, so the kernel streams the inverses at memory speed
// instead of waiting on 2m dependent substitution steps.
// WPB warps per body (CTA of 128 threads = 4 / WPB bodies): with WPB = 4 each warp takes a quarter of the
// columns and the four partial sums are added through shared memory in a fixed order -- four times as many
// loads in flight when there are too few bodies (< 2,048) to fill the GPU with one warp each.
// With `vnorm` set the input is first scaled, v = scal[rhs][1] * in (the Arnoldi normalisation v_{j+1} = w / h_{j+1,j},
// or r / beta at the start of a cycle), v is stored to vnorm as the new Krylov vector and the kernel applies P^-1
// to it: the normalisation costs no launch of its own.
template <int WPB>
__global__ void __launch_bounds__(128)
precond_apply_kernel(const void* __restrict__ precond, const double* __restrict__ in,
                     double* __restrict__ out, int64_t n_blobs, int64_t n_bodies,
                     int64_t vec_stride /* between right-hand sides (blockIdx.y) */,
                     float* __restrict__ lam32 /* optional float copy of lambda, [rhs][3 n_blobs] */,
                     const double* __restrict__ scal, double* __restrict__ vnorm,
                     const int* __restrict__ skip)
{
    __shared__ double red[WPB > 1 ? WPB : 1][128];
    rpy::pdl_enter();
    if (skip != nullptr && *skip != 0) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t p = (int64_t)blockIdx.x * (4 / WPB) + warp / WPB;
    const int part = warp % WPB;
    in += (int64_t)blockIdx.y * vec_stride; out += (int64_t)blockIdx.y * vec_stride;
    if (lam32) lam32 += (int64_t)blockIdx.y * 3 * n_blobs;
    const int64_t* hdr = static_cast<const int64_t*>(precond);
    if (hdr[0] != kMagic || hdr[1] != n_bodies || hdr[2] != n_blobs) {
        // not a preconditioner of these bodies: fail loudly -- the whole output becomes NaN
        const int64_t n = 3 * n_blobs + 6 * n_bodies;
        for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
            out[i] = __longlong_as_double(0x7ff8000000000000LL);
        return;
    }
    if (p >= n_bodies) return;                       // WPB > 1: the whole CTA (one body) returns together
    const PrecondView pv = view_of(const_cast<void*>(precond), n_bodies, n_blobs, hdr[3]);
    const int64_t b0 = pv.offsets[p];
    const int m = 3 * (int)(pv.offsets[p + 1] - b0);
    const double* __restrict__ S = pv.factors + pv.mat_off[p];
    const double* __restrict__ Y = pv.Y + b0 * 18;
    const double* __restrict__ x = in + 3 * b0;
    const double* __restrict__ y = in + 3 * n_blobs + 6 * p;
    const double sc = vnorm ? scal[(int64_t)blockIdx.y * kScal + 1] : 1.0;     // every read of x, y below is sc * (.)
    if (vnorm && part == 0) {
        double* v = vnorm + (int64_t)blockIdx.y * vec_stride;
        for (int i = lane; i < m; i += 32) v[3 * b0 + i] = sc * x[i];
        if (lane < 6) v[3 * n_blobs + 6 * p + lane] = sc * y[lane];
    }
    double* t = out + 3 * b0;

    double r[6] = {0, 0, 0, 0, 0, 0};                // every warp of the body forms r and U itself (m x 6 loads)
    for (int i = lane; i < m; i += 32) {
        const double xi = sc * x[i];
#pragma unroll
        for (int c = 0; c < 6; ++c) r[c] += Y[(size_t)i * 6 + c] * xi;
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) r[c] = warp_sum(r[c]) + sc * y[c];
    double U[6];
#pragma unroll
    for (int a = 0; a < 6; ++a) {
        double s = 0.0;
#pragma unroll
        for (int c = 0; c < 6; ++c) s += pv.Nt[(size_t)p * 36 + 6 * a + c] * r[c];
        U[a] = -s;
    }
    const int j_lo = (int)((int64_t)m * part / WPB), j_hi = (int)((int64_t)m * (part + 1) / WPB);
    for (int i0 = 0; i0 < m; i0 += 128) {
        const int i_a = i0 + lane, i_b = i_a + 32, i_c = i_a + 64, i_d = i_a + 96;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
        if (i0 + 128 <= m) {
#pragma unroll 4
            for (int j = j_lo; j < j_hi; ++j) {
                const double* row = S + (size_t)j * m;
                const double xj = sc * x[j];
                a0 += row[i_a] * xj; a1 += row[i_b] * xj; a2 += row[i_c] * xj; a3 += row[i_d] * xj;
            }
        } else {
#pragma unroll 4
            for (int j = j_lo; j < j_hi; ++j) {
                const double* row = S + (size_t)j * m;
                const double xj = sc * x[j];
                if (i_a < m) a0 += row[i_a] * xj;
                if (i_b < m) a1 += row[i_b] * xj;
                if (i_c < m) a2 += row[i_c] * xj;
                if (i_d < m) a3 += row[i_d] * xj;
            }
        }
        if (WPB == 1) {
            const int idx[4] = {i_a, i_b, i_c, i_d};
            const double acc[4] = {a0, a1, a2, a3};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (idx[k] < m) {
                    double s = acc[k];
#pragma unroll
                    for (int c = 0; c < 6; ++c) s += Y[(size_t)idx[k] * 6 + c] * U[c];
                    t[idx[k]] = s;
                    if (lam32) lam32[3 * b0 + idx[k]] = (float)s;
                }
            }
        } else {
            red[part][lane] = a0; red[part][lane + 32] = a1; red[part][lane + 64] = a2; red[part][lane + 96] = a3;
            __syncthreads();
            const int i = i0 + (int)threadIdx.x;          // one row per thread, the warps' shares in a fixed order
            if (i < m) {
                double s = red[0][threadIdx.x];
#pragma unroll
                for (int w = 1; w < WPB; ++w) s += red[w][threadIdx.x];
#pragma unroll
                for (int c = 0; c < 6; ++c) s += Y[(size_t)i * 6 + c] * U[c];
                t[i] = s;
                if (lam32) lam32[3 * b0 + i] = (float)s;
            }
            __syncthreads();
        }
    }
    if (part == 0 && lane < 6) {
        double v = U[0];
#pragma unroll
        for (int c = 1; c < 6; ++c) if (lane == c) v = U[c];
        out[3 * n_blobs + 6 * p + lane] = v;
    }
}

// ------------------------------------------------------------------ Krylov vector operations
// A solver vector has n = 3 n_blobs + 6 n_bodies doubles.  The solver runs `nrhs` independent GMRES
// processes in lockstep (one right-hand side each: blockIdx.y = right-hand side in every kernel
// below); vectors of one right-hand side are `ldv` doubles apart, Krylov vector v of right-hand side
// r is at V + (v * nrhs + r) * ldv.  A fixed grid of kVecBlocks CTAs cuts [0, n) into equal
// contiguous chunks; every reduction is two-stage (per-CTA partials, then a fixed-order sum), so the
// solve is bit-reproducible whenever the matvec is.
//
// One Arnoldi step ("GMRES"; reading A16) is seven launches:
//   precond_apply (v_j = w / h_{j,j-1} fused in), prepack, all-pairs, saddle_tail (finalise fused in),
//   dots, update (second pass's dots fused in), update (norm, Hessenberg/Givens and the convergence test
//   fused in: done by whichever CTA finishes last, in a fixed order).
// The convergence test sets ctl[0]; every kernel of a later step returns at once when it is set, so the host
// may enqueue step j+1 before it has read the outcome of step j.

__device__ __forceinline__ void chunk_of(int64_t n, int64_t& lo, int64_t& hi)
{
    const int64_t per = (n + gridDim.x - 1) / gridDim.x;
    lo = (int64_t)blockIdx.x * per;
    hi = lo + per < n ? lo + per : n;
    if (lo > n) lo = n;
}

// partial[(r * pvec + v) * gridDim.x + blk] = sum over the CTA's chunk of V[v][r][i] * w[r][i], warp w of the CTA
// takes v = w, w + 8, ...
__device__ __forceinline__ void chunk_dots(const double* __restrict__ V, int64_t ldv, int nrhs, int nvec,
                                           const double* __restrict__ wr, int64_t lo, int64_t hi,
                                           double* __restrict__ partial, int pvec)
{
    const int r = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int v = warp; v < nvec; v += kVecThreads / 32) {
        const double* a = V + ((int64_t)v * nrhs + r) * ldv;
        double s = 0.0;
        for (int64_t i = lo + lane; i < hi; i += 32) s += a[i] * wr[i];
        s = warp_sum(s);
        if (lane == 0) partial[((int64_t)r * pvec + v) * gridDim.x + blockIdx.x] = s;
    }
}

__global__ void __launch_bounds__(kVecThreads)
dots_kernel(const double* __restrict__ V, int64_t ldv, int nrhs, int nvec, const double* __restrict__ w, int64_t n,
            double* __restrict__ partial, int pvec, const int* __restrict__ skip)
{
    rpy::pdl_enter();
    if (skip != nullptr && *skip != 0) return;
    int64_t lo, hi; chunk_of(n, lo, hi);
    chunk_dots(V, ldv, nrhs, nvec, w + (int64_t)blockIdx.y * ldv, lo, hi, partial, pvec);
}

// Small state of one GMRES cycle, all on the device; every array has one slice per right-hand side
// (slice r of an array with `len` entries per right-hand side starts at r * len).
struct GmresState {
    double* R;        // [(restart+1) * restart] column-major rotated Hessenberg (upper triangular after rotation)
    double* cs;       // [restart]
    double* sn;       // [restart]
    double* g;        // [restart+1] rotated right-hand side
    double* hcol;     // [restart+1] current Hessenberg column (sum of the two Gram-Schmidt passes)
    double* yv;       // [restart]   solution of R y = g
    double* scal;     // [kScal] [0] beta or h_{j+1,j}; [1] its reciprocal; [2] |g_{j+1}|; [3] ||b||; [4] beta of this cycle
    int* ctl;         // [0] Arnoldi steps done when this cycle was told to stop (0: running); [1] converged;
                      // [2] ticket counter of the last-CTA election; [3] iterations done by the solve
    unsigned char* snap;   // [2][kSnapBytes] what the host reads after step j, in slot j & 1 (the live state may already
                           // belong to step j+1, which is enqueued before step j is read): int stop, converged,
                           // iterations, pad; then |g_{j+1}| of every right-hand side
    int restart;
};

// What the CTA that finishes an Arnoldi step last needs for the convergence test.
struct StepEnd {
    int enabled;              // 0: first Gram-Schmidt pass (no step end)
    int j;                    // step index inside the cycle
    int max_iter;
    int mixed;                // the estimates are those of the fp32 operator: end the cycle, do not declare convergence
    double tol;
    double inner_reduction;   // mixed: a cycle may reduce its start residual by this factor
    double inner_tol_factor;  // mixed: ... or reach this fraction of tol
    double f32_bound;         // mixed: relative accuracy assumed of an fp32 product (kF32ProductBound)
};

// Column j of the Hessenberg matrix of right-hand side r: hcol[0..j] from Gram-Schmidt, h_{j+1,j} = hn;
// earlier Givens rotations, the new rotation, g update (Saad & Schultz; "GMRES").  One warp: the
// lanes first stage the column and the rotations in shared memory (`stage`, 3 (restart + 2) doubles), then lane 0
// walks the chain of rotations there instead of through dependent global loads.
__device__ void hessenberg_update(const GmresState& st, int r, int j, double hn, double* stage)
{
    const int m = st.restart, ldr = m + 1, lane = threadIdx.x & 31;
    double* scal = st.scal + (int64_t)r * kScal;
    double* cs = st.cs + (int64_t)r * m; double* sn = st.sn + (int64_t)r * m;
    double* g = st.g + (int64_t)r * ldr; const double* hcol = st.hcol + (int64_t)r * ldr;
    double* col = stage; double* scs = stage + (m + 2); double* ssn = stage + 2 * (m + 2);
    for (int i = lane; i <= j; i += 32) col[i] = __ldcg(hcol + i);   // written by another CTA of this launch
    for (int i = lane; i < j; i += 32) { scs[i] = cs[i]; ssn[i] = sn[i]; }
    __syncwarp();
    if (lane == 0) {
        scal[0] = hn;
        scal[1] = hn > 0.0 ? 1.0 / hn : 0.0;
        col[j + 1] = hn;
        for (int i = 0; i < j; ++i) {
            const double t = scs[i] * col[i] + ssn[i] * col[i + 1];
            col[i + 1] = -ssn[i] * col[i] + scs[i] * col[i + 1];
            col[i] = t;
        }
        const double d = hypot(col[j], col[j + 1]);
        const double c = d > 0.0 ? col[j] / d : 1.0, sgn = d > 0.0 ? col[j + 1] / d : 0.0;
        cs[j] = c; sn[j] = sgn;
        col[j] = d; col[j + 1] = 0.0;
        const double gj = g[j];
        g[j + 1] = -sgn * gj;
        g[j] = c * gj;
        scal[2] = fabs(sgn * gj);
    }
    __syncwarp();
    double* out = st.R + (int64_t)r * ldr * m + (size_t)j * ldr;
    for (int i = lane; i <= j + 1; i += 32) out[i] = col[i];
}

// h[v] = sum_blk partial[r][v][blk] (fixed order);  w -= sum_v h[v] V[v];  norm_partial[r][blk] = |w chunk|^2;
// CTA 0 also does hcol[r][v] = (accumulate ? hcol[r][v] : 0) + h[v].
// First Gram-Schmidt pass (dots_out set): the CTA also leaves the second pass's dot products of its chunk.
// Second pass (end.enabled): the CTA that finishes last adds the norm partials of every right-hand side in a
// fixed order, h_{j+1,j} = sqrt(sum), updates the Hessenberg problems and takes the convergence decision.
__global__ void __launch_bounds__(kVecThreads)
update_kernel(const double* __restrict__ V, int64_t ldv, int nrhs, int nvec, double* __restrict__ w, int64_t n,
              const double* __restrict__ partial, int pvec, double* __restrict__ hcol, int accumulate,
              double* __restrict__ norm_partial, double* __restrict__ dots_out, GmresState st, StepEnd end,
              const int* __restrict__ skip)
{
    __shared__ double h[RPY_RIGID_MAX_RESTART + 1];
    __shared__ double red[kVecThreads / 32];
    __shared__ double stage[RPY_RIGID_MAX_BATCH][3 * (RPY_RIGID_MAX_RESTART + 2)];
    __shared__ int s_last;
    rpy::pdl_enter();
    if (skip != nullptr && *skip != 0) return;
    const int r = blockIdx.y;
    for (int v = threadIdx.x >> 5; v < nvec; v += kVecThreads / 32) {      // one warp per dot product
        double s = 0.0;
        for (int b = threadIdx.x & 31; b < (int)gridDim.x; b += 32) s += partial[((int64_t)r * pvec + v) * gridDim.x + b];
        s = warp_sum(s);
        if ((threadIdx.x & 31) == 0) {
            h[v] = s;
            if (blockIdx.x == 0) hcol[(int64_t)r * pvec + v] = (accumulate ? hcol[(int64_t)r * pvec + v] : 0.0) + s;
        }
    }
    __syncthreads();
    int64_t lo, hi; chunk_of(n, lo, hi);
    double* wr = w + (int64_t)r * ldv;
    double nrm = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += kVecThreads) {
        double wi = wr[i];
        for (int v = 0; v < nvec; ++v) wi -= h[v] * V[((int64_t)v * nrhs + r) * ldv + i];
        wr[i] = wi;
        nrm += wi * wi;
    }
    nrm = warp_sum(nrm);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = nrm;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < kVecThreads / 32; ++k) s += red[k];
        norm_partial[(int64_t)r * gridDim.x + blockIdx.x] = s;
    }
    if (dots_out) chunk_dots(V, ldv, nrhs, nvec, wr, lo, hi, dots_out, pvec);    // after the barrier: the chunk of w is final
    if (!end.enabled) return;

    // ---- end of the Arnoldi step: the last CTA to get here closes it
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&st.ctl[2], 1) == (int)(gridDim.x * gridDim.y) - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp < nrhs) {                                   // nrhs <= RPY_RIGID_MAX_BATCH = warps of the CTA
        double s = 0.0;                                  // fixed-order strided sums, then shuffles
        for (int b = lane; b < (int)gridDim.x; b += 32) s += __ldcg(norm_partial + (int64_t)warp * gridDim.x + b);
        s = warp_sum(s);
        hessenberg_update(st, warp, end.j, sqrt(s), stage[warp]);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        bool all_conv = true, inner_all = true, all_certified = true;
        for (int q = 0; q < nrhs; ++q) {
            const double* sc = st.scal + (int64_t)q * kScal;
            const double res = sc[2], bn = sc[3];
            const double rel = bn > 0.0 ? res / bn : 0.0;
            if (rel > end.tol) all_conv = false;
            // mixed: the cycle started from a TRUE residual sc[4]; with products of relative accuracy f32_bound the
            // true residual now is within margin = f32_bound * sc[4] / |b| of the estimate (inexact Krylov, PAPER.md:222
            // [79]).  Once that margin is small against tol the cycle runs to tol - margin and the solve is over
            // without another fp64 product; before that it ends after inner_reduction and the fp64 residual decides.
            const double margin = bn > 0.0 ? end.f32_bound * sc[4] / bn : 0.0;
            const bool certifiable = margin <= 0.5 * end.tol;
            if (certifiable) {
                if (rel > end.tol - margin) { all_certified = false; inner_all = false; }
            } else {
                all_certified = false;
                // the cycle's own goal: inner_reduction, or -- when that is within a factor 4 -- the level from which the
                // NEXT cycle can be certified (tol / (2 f32_bound)), so that the solve ends there
                double level = end.inner_reduction * sc[4];
                const double cert_level = 0.5 * end.tol / end.f32_bound * bn;
                if (cert_level < level && cert_level >= 0.25 * level) level = cert_level;
                if (rel > end.inner_tol_factor * end.tol && res > level) inner_all = false;
            }
        }
        const int n_iter = st.ctl[3] + 1;
        st.ctl[3] = n_iter;
        st.ctl[2] = 0;
        if (end.mixed) {
            if (inner_all || n_iter >= end.max_iter) {
                st.ctl[0] = end.j + 1;
                st.ctl[1] = all_certified ? 1 : 0;
            }
        } else if (all_conv || n_iter >= end.max_iter) {
            st.ctl[0] = end.j + 1;
            st.ctl[1] = all_conv ? 1 : 0;
        }
        int* si = reinterpret_cast<int*>(st.snap + (size_t)(end.j & 1) * kSnapBytes);
        double* sr = reinterpret_cast<double*>(si + 4);
        si[0] = st.ctl[0]; si[1] = st.ctl[1]; si[2] = n_iter; si[3] = 0;
        for (int q = 0; q < nrhs; ++q) sr[q] = st.scal[(int64_t)q * kScal + 2];
    }
}

// beta = sqrt(sum partial) at the start of a cycle: g = (beta, 0, ...), scal[0..1] = beta, 1/beta, scal[4] = beta;
// with set_bnorm, scal[3] = beta (the first cycle starts from x0 = 0, so r0 = b) and the iteration count is
// cleared.  The cycle's stop flag is cleared.
__global__ void cycle_start_kernel(GmresState st, const double* __restrict__ norm_partial, int nblk, int set_bnorm)
{
    rpy::pdl_enter();
    const int r = blockIdx.x, ldr = st.restart + 1;
    double s = 0.0;
    for (int b = threadIdx.x; b < nblk; b += 32) s += norm_partial[(int64_t)r * nblk + b];
    s = warp_sum(s);
    if (threadIdx.x != 0) return;
    double* scal = st.scal + (int64_t)r * kScal;
    double* g = st.g + (int64_t)r * ldr;
    const double beta = sqrt(s);
    scal[0] = beta; scal[1] = beta > 0.0 ? 1.0 / beta : 0.0; scal[2] = beta; scal[4] = beta;
    if (set_bnorm) scal[3] = beta;
    for (int i = 0; i < ldr; ++i) g[i] = i == 0 ? beta : 0.0;
    if (r == 0) {
        st.ctl[0] = 0; st.ctl[1] = 0; st.ctl[2] = 0;
        if (set_bnorm) st.ctl[3] = 0;
    }
}

// R y = g for the first k columns (back substitution); a zero pivot (a right-hand side that was
// already solved exactly, or a zero right-hand side) gives y_i = 0.
__global__ void solve_y_kernel(GmresState st, int k)
{
    rpy::pdl_enter();
    if (threadIdx.x != 0) return;
    const int r = blockIdx.x, m = st.restart, ldr = m + 1;
    const double* R = st.R + (int64_t)r * ldr * m; const double* g = st.g + (int64_t)r * ldr;
    double* yv = st.yv + (int64_t)r * m;
    for (int i = k - 1; i >= 0; --i) {
        double s = g[i];
        for (int c = i + 1; c < k; ++c) s -= R[(size_t)c * ldr + i] * yv[c];
        const double piv = R[(size_t)i * ldr + i];
        yv[i] = piv != 0.0 ? s / piv : 0.0;
    }
}

// out[r][i] = sum_{v<k} y[r][v] V[v][r][i]
__global__ void combine_kernel(const double* __restrict__ V, int64_t ldv, int nrhs, int k, const double* __restrict__ y,
                               int ylen, double* __restrict__ out, int64_t n)
{
    rpy::pdl_enter();
    const int r = blockIdx.y;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int v = 0; v < k; ++v) s += y[(int64_t)r * ylen + v] * V[((int64_t)v * nrhs + r) * ldv + i];
        out[(int64_t)r * ldv + i] = s;
    }
}

// y[r][i] = alpha * x[r][i] + beta * y[r][i]   (beta == 0 overwrites)
__global__ void axpby_kernel(double alpha, const double* __restrict__ x, int64_t x_stride, double beta,
                             double* __restrict__ y, int64_t y_stride, int64_t n)
{
    rpy::pdl_enter();
    const double* xr = x + (int64_t)blockIdx.y * x_stride; double* yr = y + (int64_t)blockIdx.y * y_stride;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        yr[i] = beta == 0.0 ? alpha * xr[i] : alpha * xr[i] + beta * yr[i];
}

// |w[r] chunk|^2 per CTA (the norm of a vector through the same two-stage reduction)
__global__ void __launch_bounds__(kVecThreads)
norm_partial_kernel(const double* __restrict__ w, int64_t ldv, int64_t n, double* __restrict__ norm_partial)
{
    __shared__ double red[kVecThreads / 32];
    rpy::pdl_enter();
    const double* wr = w + (int64_t)blockIdx.y * ldv;
    int64_t lo, hi; chunk_of(n, lo, hi);
    double nrm = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += kVecThreads) nrm += wr[i] * wr[i];
    nrm = warp_sum(nrm);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = nrm;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < kVecThreads / 32; ++k) s += red[k];
        norm_partial[(int64_t)blockIdx.y * gridDim.x + blockIdx.x] = s;
    }
}

__global__ void to_float_kernel(const double* __restrict__ in, int64_t in_stride, float* __restrict__ out, int64_t out_stride, int64_t n,
                                const int* __restrict__ skip = nullptr)
{
    rpy::pdl_enter();
    if (skip != nullptr && *skip != 0) return;
    const double* a = in + (int64_t)blockIdx.y * in_stride; float* o = out + (int64_t)blockIdx.y * out_stride;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) o[i] = (float)a[i];
}

}  // namespace

// =================================================================== host side
namespace {

// mat_off[p] = sum_{p' < p} (3 blobs_{p'})^2 (exclusive scan, one CTA of 1024 threads), mat_off[nb] = total.
__global__ void matoff_kernel(const int64_t* __restrict__ off, int64_t* __restrict__ mo, int64_t nb)
{
    __shared__ long long wsum[32];
    __shared__ long long carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int64_t base = 0; base < nb; base += 1024) {
        const int64_t i = base + tid;
        long long v = 0;
        if (i < nb) { const long long m = 3 * (off[i + 1] - off[i]); v = m * m; }
        long long incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const long long t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            long long w = wsum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const long long t = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += t; }
            wsum[lane] = w;                          // inclusive sums of the warps' totals
        }
        __syncthreads();
        const long long before = carry + (warp > 0 ? wsum[warp - 1] : 0);
        if (i < nb) mo[i] = before + incl - v;
        __syncthreads();
        if (tid == 0) carry += wsum[31];
        __syncthreads();
    }
    if (tid == 0) mo[nb] = carry;
}

inline bool finite_pos(double v) { return v > 0.0 && isfinite(v); }
inline unsigned warp_grid(int64_t n_bodies, int threads) { return (unsigned)((n_bodies * 32 + threads - 1) / threads); }

#define RPY_CUDA_TRY(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) return rpy::set_cuda_error(e__); } while (0)

rpy_status check_bodies(int64_t n_blobs, int64_t n_bodies)
{
    if (n_blobs < 0 || n_blobs > RPY_MAX_BLOBS || n_bodies < 0 || n_bodies > n_blobs) return RPY_ERR_ARG;
    return RPY_OK;
}

constexpr rpy_prec kPrecMixed = static_cast<rpy_prec>(RPY_PREC_MIXED);
// Mixed solve (reading A21): a cycle of fp32 products ends once its residual estimate has fallen by
// kInnerReduction or is below kInnerTolFactor * tol; the fp64 residual of the restart then decides.  Measured
// (B200, tol 1e-8): 1e-4 / 1.0 needs 45 (cfg 2) and 23 (cfg 3) iterations and two fp64 products; a deeper
// first cycle with a safety margin on the second (1e-5 / 0.5) needs 47 and 25 iterations for the same two
// fp64 products -- every restart discards the Krylov space, so the shallower split wins.
constexpr double kInnerReduction = 1e-4;
constexpr double kInnerTolFactor = 1.0;
// What a cycle of fp32 products can do to the residual behind the back of its Arnoldi estimate, relative to the TRUE
// residual rho the cycle started from (fp64 product): |true - estimate| <= kF32ProductBound * rho.  "Krylov methods allow
// one to lower the accuracy of the matrix-vector product as the residual is reduced" ([79]): the gap is the
// product's error on the cycle's correction, <= (a few eps_fp32) |M| |d lambda| <= (a few eps_fp32) cond(M) rho, i.e. ~6e-5 rho
// for cond(M) ~ 1e3 (pin P4: the smallest eigenvalue of M is 0.04-0.07 of the largest).  Measured on cfg 2 / cfg 3 / the
// Table III rods, cycles 1 and 2: 0.3e-5 ... 2.2e-5.  With 1e-4: once kF32ProductBound * rho <= tol / 2 a cycle runs to
// tol - margin and no further fp64 product is spent on confirming it; what is reported then is estimate + margin, an upper
// bound.  tol = 1e-8: cycle 1 to 5e-5 (fp64 residual), cycle 2 to the end: ONE fp64 product instead of two.
constexpr double kF32ProductBound = 1e-4;

// Solver workspace, carved from one caller-owned buffer (nrhs lockstep right-hand sides).
struct SolveWs {
    int64_t n; size_t vec_bytes; int nrhs;
    double *V, *w, *z, *x, *b;
    GmresState st;
    double *partial, *partial2, *norm_partial;
    unsigned char* status;            // [64 bytes: ctl ints][kScal doubles per right-hand side]: one read-back
    float *pos32, *lam32, *vel32;
    void* mv; size_t mv_bytes;
    size_t total;
};

size_t mv_bytes_of(rpy_prec prec, int64_t n_blobs, int nrhs)
{
    // every solve also forms fp64 residuals (the mixed solve per cycle, the fp32 solve once at the end)
    if (prec == RPY_PREC_F64) return rpy_matvec_workspace_bytes(prec, n_blobs, nrhs);
    const size_t a = rpy_matvec_workspace_bytes(RPY_PREC_F64, n_blobs, nrhs), b = rpy_matvec_workspace_bytes(RPY_PREC_F32_ACC64, n_blobs, nrhs);
    return a > b ? a : b;
}

SolveWs carve(rpy_prec prec, int64_t n_blobs, int64_t n_bodies, int restart, int nrhs, void* base)
{
    SolveWs W;
    unsigned char* p = static_cast<unsigned char*>(base);
    size_t at = 0;
    auto take = [&](size_t bytes) { unsigned char* r = p ? p + at : nullptr; at = align_up(at + bytes, kAlign); return r; };
    const size_t k = (size_t)nrhs;
    W.nrhs = nrhs;
    W.n = 3 * n_blobs + 6 * n_bodies;
    W.vec_bytes = align_up((size_t)W.n * 8, kAlign);
    W.V = (double*)take(W.vec_bytes * (size_t)(restart + 1) * k);
    W.w = (double*)take(W.vec_bytes * k); W.z = (double*)take(W.vec_bytes * k);
    W.x = (double*)take(W.vec_bytes * k); W.b = (double*)take(W.vec_bytes * k);
    W.st.restart = restart;
    W.st.R = (double*)take((size_t)(restart + 1) * restart * 8 * k);
    W.st.cs = (double*)take((size_t)restart * 8 * k); W.st.sn = (double*)take((size_t)restart * 8 * k);
    W.st.g = (double*)take((size_t)(restart + 1) * 8 * k); W.st.hcol = (double*)take((size_t)(restart + 1) * 8 * k);
    W.st.yv = (double*)take((size_t)restart * 8 * k);
    W.status = take(64 + (size_t)kScal * 8 * k);
    W.st.ctl = (int*)W.status; W.st.scal = (double*)(p ? W.status + 64 : nullptr);
    W.st.snap = take(2 * kSnapBytes);
    W.partial = (double*)take((size_t)kVecBlocks * (restart + 1) * 8 * k);
    W.partial2 = (double*)take((size_t)kVecBlocks * (restart + 1) * 8 * k);
    W.norm_partial = (double*)take((size_t)kVecBlocks * 8 * k);
    if (prec != RPY_PREC_F64) {
        W.pos32 = (float*)take((size_t)n_blobs * 12); W.lam32 = (float*)take((size_t)n_blobs * 12 * k);
        W.vel32 = (float*)take((size_t)n_blobs * 12 * k);
    } else { W.pos32 = W.lam32 = W.vel32 = nullptr; }
    W.mv_bytes = mv_bytes_of(prec, n_blobs, nrhs);
    W.mv = take(W.mv_bytes);
    W.total = at;
    return W;
}

inline int64_t vec_stride(const SolveWs& W) { return (int64_t)(W.vec_bytes / 8); }
inline dim3 vgrid(int nrhs) { return dim3(kVecBlocks, (unsigned)nrhs); }

// How one rank's share of the product is completed (include/rpy_rigid.h, rpy_rigid_solve_ext).
struct ShardCtx { int shard = 0, n_shards = 1; rpy_reduce_fn reduce = nullptr; void* ctx = nullptr; };

// out[r] = [M lambda_r - K U_r ; -K^T lambda_r] for the nrhs solver vectors in[r] (stride `stride`):
// Eq. (11)'s operator; ONE product call with n_rhs = nrhs.  pos32 must hold float(pos) for the fp32 product.
// skip: device flag that turns the whole application into a no-op (see "Krylov vector operations").
rpy_status saddle(int wall, rpy_prec prec, int64_t N, int64_t nb, const double* pos, const double* q,
                  const int64_t* off, double a, double eta, const double* in, double* out, int64_t stride,
                  int nrhs, const SolveWs& W, cudaStream_t st, bool lam32_ready = false, const int* skip = nullptr,
                  const ShardCtx& sh = ShardCtx{})
{
    rpy_status s;
    const bool f64 = prec == RPY_PREC_F64;
    if (!f64 && !lam32_ready)
        RPY_CUDA_TRY(rpy::launch_pdl(to_float_kernel, vgrid(nrhs), dim3(256), 0, st, in, stride, W.lam32, 3 * N, 3 * N, skip));
    const void* mpos = f64 ? (const void*)pos : (const void*)W.pos32;
    const void* mforce = f64 ? (const void*)in : (const void*)W.lam32;
    const int64_t fstride = f64 ? stride : 3 * N;
    const dim3 bg(warp_grid(nb, 128), (unsigned)nrhs);
    rpy::PartialSums ps{nullptr, 0, 0, 0.0};
    if (sh.n_shards > 1) {
        // this rank's share of the unordered pairs, as doubles, straight into out; the caller's hook adds the ranks
        s = rpy::matvec_strided(wall != 0, prec, N, nrhs, mpos, mforce, fstride, out, stride, a, eta, W.mv, W.mv_bytes, st,
                                skip, nullptr, sh.shard, sh.n_shards, true);
        if (s != RPY_OK) return s;
        if (sh.reduce(sh.ctx, out, 3 * N, st) != 0) return RPY_ERR_ARG;
        RPY_CUDA_TRY(rpy::launch_pdl(saddle_tail_kernel, bg, dim3(128), 0, st, pos, q, off, in, (const float*)nullptr, out, N, nb, stride, ps, skip));
    } else if (nrhs == 1 || nrhs == 2 || nrhs == 4 || nrhs == 8) {
        // one right-hand-side group: the product stops before its finalise step, the tail adds the slices
        s = rpy::matvec_strided(wall != 0, prec, N, nrhs, mpos, mforce, fstride, nullptr, 0, a, eta, W.mv, W.mv_bytes, st,
                                skip, &ps);
        if (s != RPY_OK) return s;
        RPY_CUDA_TRY(rpy::launch_pdl(saddle_tail_kernel, bg, dim3(128), 0, st, pos, q, off, in, (const float*)nullptr, out, N, nb, stride, ps, skip));
    } else if (f64) {
        s = rpy::matvec_strided(wall != 0, prec, N, nrhs, pos, in, stride, out, stride, a, eta, W.mv, W.mv_bytes, st, skip);
        if (s != RPY_OK) return s;
        RPY_CUDA_TRY(rpy::launch_pdl(saddle_tail_kernel, bg, dim3(128), 0, st, pos, q, off, in, (const float*)nullptr, out, N, nb, stride, ps, skip));
    } else {
        s = rpy::matvec_strided(wall != 0, prec, N, nrhs, W.pos32, W.lam32, 3 * N, W.vel32, 3 * N, a, eta, W.mv, W.mv_bytes, st, skip);
        if (s != RPY_OK) return s;
        RPY_CUDA_TRY(rpy::launch_pdl(saddle_tail_kernel, bg, dim3(128), 0, st, pos, q, off, in, (const float*)W.vel32, out, N, nb, stride, ps, skip));
    }
    RPY_CUDA_TRY(cudaGetLastError());
    return RPY_OK;
}

// [lambda; U] = P^-1 in; with `vnorm` the input is first scaled by scal[rhs][1] and stored there (see the kernel).
rpy_status precond_apply(int64_t N, int64_t nb, const void* precond, const double* in, double* out, int64_t stride,
                         int nrhs, cudaStream_t st, float* lam32 = nullptr, const double* scal = nullptr,
                         double* vnorm = nullptr, const int* skip = nullptr)
{
    // one warp per body streams the inverses at HBM speed once there are enough bodies (cfg 3, 4,096 bodies:
    // 0.099 ms = 5.9 TB/s against 0.120 ms with four); below ~14 warps per SM four warps per body (a CTA each)
    // keep more loads in flight (cfg 2, 1,000 bodies: 14 against 30 us cold)
    if (nb >= 2048)
        RPY_CUDA_TRY(rpy::launch_pdl(precond_apply_kernel<1>, dim3(warp_grid(nb, 128), (unsigned)nrhs), dim3(128), 0, st,
                                     precond, in, out, N, nb, stride, lam32, scal, vnorm, skip));
    else
        RPY_CUDA_TRY(rpy::launch_pdl(precond_apply_kernel<4>, dim3((unsigned)nb, (unsigned)nrhs), dim3(128), 0, st,
                                     precond, in, out, N, nb, stride, lam32, scal, vnorm, skip));
    RPY_CUDA_TRY(cudaGetLastError());
    return RPY_OK;
}

}  // namespace

extern "C" {

rpy_status rpy_rigid_K_apply(int64_t n_blobs, int64_t n_bodies, const double* d_pos, const double* d_q,
                             const int64_t* d_offsets, const double* d_U, double alpha, double beta,
                             double* d_out, void* cuda_stream)
{
    rpy_status s = check_bodies(n_blobs, n_bodies);
    if (s != RPY_OK) return s;
    if (n_blobs == 0 || n_bodies == 0) return RPY_OK;
    if (!d_pos || !d_q || !d_offsets || !d_U || !d_out) return RPY_ERR_NULL;
    if (!isfinite(alpha) || !isfinite(beta)) return RPY_ERR_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    k_apply_kernel<<<warp_grid(n_bodies, 128), 128, 0, st>>>(d_pos, d_q, d_offsets, d_U, alpha, beta, d_out, n_bodies, 0, 0);
    RPY_CUDA_TRY(cudaGetLastError());
    return RPY_OK;
}

rpy_status rpy_rigid_KT_apply(int64_t n_blobs, int64_t n_bodies, const double* d_pos, const double* d_q,
                              const int64_t* d_offsets, const double* d_lambda, double alpha, double beta,
                              double* d_out, void* cuda_stream)
{
    rpy_status s = check_bodies(n_blobs, n_bodies);
    if (s != RPY_OK) return s;
    if (n_blobs == 0 || n_bodies == 0) return RPY_OK;
    if (!d_pos || !d_q || !d_offsets || !d_lambda || !d_out) return RPY_ERR_NULL;
    if (!isfinite(alpha) || !isfinite(beta)) return RPY_ERR_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    kt_apply_kernel<<<warp_grid(n_bodies, 128), 128, 0, st>>>(d_pos, d_q, d_offsets, d_lambda, alpha, beta, d_out, n_bodies, 0, 0);
    RPY_CUDA_TRY(cudaGetLastError());
    return RPY_OK;
}

rpy_status rpy_rigid_blob_positions(rpy_prec prec, int64_t n_bodies, int blobs_per_body, const void* d_template,
                                    const void* d_centres, const void* d_quats, void* d_pos, void* cuda_stream)
{
    if (prec != RPY_PREC_F64 && prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    if (n_bodies < 0 || blobs_per_body < 1 || n_bodies * (int64_t)blobs_per_body > RPY_MAX_BLOBS) return RPY_ERR_ARG;
    if (n_bodies == 0) return RPY_OK;
    if (!d_template || !d_centres || !d_quats || !d_pos) return RPY_ERR_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int64_t total = n_bodies * blobs_per_body;
    const unsigned blocks = (unsigned)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
    if (prec == RPY_PREC_F64)
        blob_positions_kernel<double><<<blocks, 256, 0, st>>>((const double*)d_template, (const double*)d_centres,
                                                             (const double*)d_quats, (double*)d_pos, n_bodies, blobs_per_body);
    else
        blob_positions_kernel<float><<<blocks, 256, 0, st>>>((const float*)d_template, (const float*)d_centres,
                                                            (const float*)d_quats, (float*)d_pos, n_bodies, blobs_per_body);
    RPY_CUDA_TRY(cudaGetLastError());
    return RPY_OK;
}

size_t rpy_rigid_precond_bytes(int64_t n_bodies, const int64_t* h_offsets)
{
    PrecondLayout L;
    if (!layout_of(n_bodies, h_offsets, L) || L.n_blobs > RPY_MAX_BLOBS) return 0;
    return L.total;
}

rpy_status rpy_rigid_precond_build(int wall, int64_t n_blobs, int64_t n_bodies, const double* d_pos,
                                   const double* d_q, const int64_t* h_offsets, double a, double eta,
                                   void* d_precond, size_t precond_bytes, void* cuda_stream)
{
    rpy_status s = check_bodies(n_blobs, n_bodies);
    if (s != RPY_OK) return s;
    if (!finite_pos(a) || !finite_pos(eta)) return RPY_ERR_ARG;
    if (n_bodies == 0) return n_blobs == 0 ? RPY_OK : RPY_ERR_ARG;
    if (!d_pos || !d_q || !h_offsets || !d_precond) return RPY_ERR_NULL;
    PrecondLayout L;
    if (!layout_of(n_bodies, h_offsets, L) || L.n_blobs != n_blobs) return RPY_ERR_ARG;
    if (precond_bytes < L.total || ((uintptr_t)d_precond % kAlign) != 0) return RPY_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // tables: header (4 words), the caller's offsets copied up as they are, matrix offsets scanned on the device
    const int64_t hdr[kHdrWords] = {kMagic, n_bodies, n_blobs, L.total_mat, -1};
    // bodies with 3 n_p <= kRegMaxM: the register-resident sweep; larger ones: the shared/global-memory Cholesky
    size_t smem = 0;
    int max_small = 0;
    bool any_big = false;
    for (int64_t p = 0; p < n_bodies; ++p) {
        const int64_t m = 3 * (h_offsets[p + 1] - h_offsets[p]);
        if (m <= kRegMaxM) { if (m > max_small) max_small = (int)m; continue; }
        any_big = true;
        if (m <= kSmemBodyM) { size_t need = ((size_t)(m | 1) * m + 6 * m) * 8; if (need > smem) smem = need; }
    }
    unsigned char* base = static_cast<unsigned char*>(d_precond);
    RPY_CUDA_TRY(cudaMemcpyAsync(base, hdr, sizeof hdr, cudaMemcpyHostToDevice, st));
    RPY_CUDA_TRY(cudaMemcpyAsync(base + L.offsets_at, h_offsets, (size_t)(n_bodies + 1) * 8, cudaMemcpyHostToDevice, st));
    RPY_CUDA_TRY(cudaStreamSynchronize(st));      // hdr and h_offsets have been read: both may go away now
    matoff_kernel<<<1, 1024, 0, st>>>(reinterpret_cast<const int64_t*>(base + L.offsets_at),
                                     reinterpret_cast<int64_t*>(base + L.matoff_at), n_bodies);
    PrecondView v = view_of(d_precond, n_bodies, n_blobs, L.total_mat);
    const double PI = 3.14159265358979323846;
    const double scale = 1.0 / (6.0 * PI * eta * a);
    if (max_small > 0) {
        const int TA = (max_small + kRT - 1) / kRT + 1;
        const int threads = (TA * (TA + 1) / 2 + 31) / 32 * 32;
        // 22 KB of panels per CTA: ask for a carve-out that lets the register-limited two CTAs per SM in
        RPY_CUDA_TRY(cudaFuncSetAttribute(precond_build_reg_kernel<true>, cudaFuncAttributePreferredSharedMemoryCarveout, 50));
        RPY_CUDA_TRY(cudaFuncSetAttribute(precond_build_reg_kernel<false>, cudaFuncAttributePreferredSharedMemoryCarveout, 50));
        if (wall) precond_build_reg_kernel<true><<<(unsigned)n_bodies, threads, 0, st>>>(d_pos, d_q, v.offsets, v.mat_off, v.info,
                                                                                       v.factors, v.Y, v.Nt, 1.0 / a, scale);
        else      precond_build_reg_kernel<false><<<(unsigned)n_bodies, threads, 0, st>>>(d_pos, d_q, v.offsets, v.mat_off, v.info,
                                                                                        v.factors, v.Y, v.Nt, 1.0 / a, scale);
        RPY_CUDA_TRY(cudaGetLastError());
        ntilde_kernel<<<(unsigned)((n_bodies + 127) / 128), 128, 0, st>>>(v.offsets, v.info, v.Nt, n_bodies, 1.0 / a);
        RPY_CUDA_TRY(cudaGetLastError());
    }
    if (any_big) {
        const int only_above = max_small > 0 ? kRegMaxM : 0;
        if (wall) {
            RPY_CUDA_TRY(cudaFuncSetAttribute(precond_build_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            precond_build_kernel<true><<<(unsigned)n_bodies, kBuildThreads, smem, st>>>(d_pos, d_q, v.offsets, v.mat_off, v.info,
                                                                                      v.factors, v.Y, v.Nt, 1.0 / a, scale, only_above);
        } else {
            RPY_CUDA_TRY(cudaFuncSetAttribute(precond_build_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            precond_build_kernel<false><<<(unsigned)n_bodies, kBuildThreads, smem, st>>>(d_pos, d_q, v.offsets, v.mat_off, v.info,
                                                                                       v.factors, v.Y, v.Nt, 1.0 / a, scale, only_above);
        }
    }
    RPY_CUDA_TRY(cudaGetLastError());
    precond_finish_kernel<<<1, 256, 0, st>>>(v.info, n_bodies, reinterpret_cast<int64_t*>(base));
    RPY_CUDA_TRY(cudaGetLastError());
    return RPY_OK;
}

}  // extern "C"

namespace {

// Copies the header down (read-only) and checks that it is a preconditioner of these bodies; *h_first = the
// first body whose factorisation failed, else -1.  n_blobs < 0: not checked (rpy_rigid_precond_info).
rpy_status first_bad(int64_t n_bodies, int64_t n_blobs, const void* precond, int64_t* h_first, cudaStream_t st)
{
    int64_t hdr[kHdrWords] = {0, 0, 0, 0, 0};
    RPY_CUDA_TRY(cudaMemcpyAsync(hdr, precond, sizeof hdr, cudaMemcpyDeviceToHost, st));
    RPY_CUDA_TRY(cudaStreamSynchronize(st));
    *h_first = -1;
    if (hdr[0] != kMagic || hdr[1] != n_bodies || (n_blobs >= 0 && hdr[2] != n_blobs)) return RPY_ERR_ARG;
    *h_first = hdr[4];
    return hdr[4] < 0 ? RPY_OK : st_of(RPY_ERR_NOT_SPD);
}

}  // namespace

extern "C" {

rpy_status rpy_rigid_precond_info(int64_t n_bodies, const void* d_precond, int64_t* h_first_bad_body, void* cuda_stream)
{
    if (n_bodies < 1) return RPY_ERR_ARG;
    if (!d_precond || !h_first_bad_body) return RPY_ERR_NULL;
    return first_bad(n_bodies, -1, d_precond, h_first_bad_body, static_cast<cudaStream_t>(cuda_stream));
}

rpy_status rpy_rigid_precond_apply(int64_t n_blobs, int64_t n_bodies, const void* d_precond,
                                   const double* d_in, double* d_out, void* cuda_stream)
{
    rpy_status s = check_bodies(n_blobs, n_bodies);
    if (s != RPY_OK) return s;
    if (n_bodies == 0) return RPY_OK;
    if (!d_precond || !d_in || !d_out) return RPY_ERR_NULL;
    const size_t bytes = (size_t)(3 * n_blobs + 6 * n_bodies) * 8;
    const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
    if (a < b + bytes && b < a + bytes) return RPY_ERR_ALIAS;
    return precond_apply(n_blobs, n_bodies, d_precond, d_in, d_out, 0, 1, static_cast<cudaStream_t>(cuda_stream));
}

rpy_status rpy_rigid_precond_get(int64_t n_bodies, const int64_t* h_offsets, const void* d_precond, int64_t body,
                                 double* d_factor, double* d_body_mobility, void* cuda_stream)
{
    if (!h_offsets || !d_precond) return RPY_ERR_NULL;
    PrecondLayout L;
    if (!layout_of(n_bodies, h_offsets, L) || body < 0 || body >= n_bodies) return RPY_ERR_ARG;
    PrecondView v = view_of(const_cast<void*>(d_precond), n_bodies, L.n_blobs, L.total_mat);
    int64_t mo = 0;
    for (int64_t p = 0; p < body; ++p) { int64_t m = 3 * (h_offsets[p + 1] - h_offsets[p]); mo += m * m; }
    const int64_t m = 3 * (h_offsets[body + 1] - h_offsets[body]);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (d_factor) RPY_CUDA_TRY(cudaMemcpyAsync(d_factor, v.factors + mo, (size_t)m * m * 8, cudaMemcpyDeviceToDevice, st));
    if (d_body_mobility) RPY_CUDA_TRY(cudaMemcpyAsync(d_body_mobility, v.Nt + body * 36, 36 * 8, cudaMemcpyDeviceToDevice, st));
    return RPY_OK;
}

size_t rpy_rigid_solve_workspace_bytes(rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies, int restart)
{
    return rpy_rigid_solve_batch_workspace_bytes(matvec_prec, n_blobs, n_bodies, restart, 1);
}

size_t rpy_rigid_solve_batch_workspace_bytes(rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies, int restart, int n_rhs)
{
    if (matvec_prec != RPY_PREC_F64 && matvec_prec != RPY_PREC_F32_ACC64 && matvec_prec != kPrecMixed) return 0;
    if (check_bodies(n_blobs, n_bodies) != RPY_OK || n_bodies < 1 || restart < 1 || restart > RPY_RIGID_MAX_RESTART) return 0;
    if (n_rhs < 1 || n_rhs > RPY_RIGID_MAX_BATCH) return 0;
    return carve(matvec_prec, n_blobs, n_bodies, restart, n_rhs, nullptr).total;
}

rpy_status rpy_rigid_saddle_apply(int wall, rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies,
                                  const double* d_pos, const double* d_q, const int64_t* d_offsets,
                                  double a, double eta, const double* d_in, double* d_out,
                                  void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (matvec_prec != RPY_PREC_F64 && matvec_prec != RPY_PREC_F32_ACC64) return RPY_ERR_ARG;
    rpy_status s = check_bodies(n_blobs, n_bodies);
    if (s != RPY_OK || n_bodies < 1) return RPY_ERR_ARG;
    if (!finite_pos(a) || !finite_pos(eta)) return RPY_ERR_ARG;
    if (!d_pos || !d_q || !d_offsets || !d_in || !d_out || !d_workspace) return RPY_ERR_NULL;
    SolveWs W = carve(matvec_prec, n_blobs, n_bodies, 1, 1, d_workspace);
    if (workspace_bytes < W.total || ((uintptr_t)d_workspace % kAlign) != 0) return RPY_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (matvec_prec == RPY_PREC_F32_ACC64) to_float_kernel<<<vgrid(1), 256, 0, st>>>(d_pos, 0, W.pos32, 0, 3 * n_blobs);
    return saddle(wall, matvec_prec, n_blobs, n_bodies, d_pos, d_q, d_offsets, a, eta, d_in, d_out, W.n, 1, W, st);
}

}  // extern "C"

namespace {

// nrhs GMRES processes in lockstep (one per right-hand side, sharing every kernel launch and ONE
// product call with n_rhs = nrhs per iteration); nrhs = 1 is the plain solve.
//
// Host and device.  The device decides: the kernel that closes Arnoldi step j applies the stopping rule and sets
// ctl[0]; the kernels of every later step return at once when it is set.  The host therefore enqueues step j+1
// BEFORE it reads the outcome of step j (the 16 + 64 nrhs bytes of W.status), and reads it on the caller's side
// stream, ordered after step j by the caller's event: the read-back and the host's launch work are covered by
// device work, and a step enqueued in vain costs seven empty kernels.  Without a side stream the host reads on
// the main stream and the device idles while the next step is being enqueued.
rpy_status solve_batch(int wall, rpy_prec matvec_prec, int64_t N, int64_t nb, int nrhs,
                       const double* d_pos, const double* d_q, const int64_t* d_offsets,
                       const double* d_F, const double* d_slip, double a, double eta,
                       const void* d_precond, double tol, int restart, int max_iter,
                       double* d_lambda, double* d_U, double* h_history, int* h_n_iter, double* h_rel_resid,
                       void* d_workspace, size_t workspace_bytes, cudaStream_t st, const rpy_rigid_solve_ext* ext)
{
    const bool mixed = matvec_prec == kPrecMixed;
    const rpy_prec inner_prec = mixed ? RPY_PREC_F32_ACC64 : matvec_prec;     // the product inside Arnoldi
    const rpy_prec outer_prec = mixed ? RPY_PREC_F64 : matvec_prec;           // the product of a restart's residual
    SolveWs W = carve(matvec_prec, N, nb, restart, nrhs, d_workspace);
    if (workspace_bytes < W.total || ((uintptr_t)d_workspace % kAlign) != 0) return RPY_ERR_WORKSPACE;
    ShardCtx sh;
    cudaStream_t side = nullptr; cudaEvent_t side_ev = nullptr;
    if (ext) {
        if (ext->n_shards < 1 || ext->shard < 0 || ext->shard >= ext->n_shards) return RPY_ERR_ARG;
        if (ext->n_shards > 1) {
            if (!ext->reduce) return RPY_ERR_NULL;
            if (nrhs != 1 || !rpy::matvec_shardable(N)) return RPY_ERR_ARG;
            sh.shard = ext->shard; sh.n_shards = ext->n_shards; sh.reduce = ext->reduce; sh.ctx = ext->reduce_ctx;
        }
        if (ext->side_stream && ext->side_event) {
            side = static_cast<cudaStream_t>(ext->side_stream); side_ev = static_cast<cudaEvent_t>(ext->side_event);
        }
    }
    const int64_t n = W.n, ldv = vec_stride(W);
    const int pvec = restart + 1;
    const dim3 vg = vgrid(nrhs);
    float* const lam32_in_cycle = inner_prec == RPY_PREC_F64 ? nullptr : W.lam32;   // P^-1 also writes float(lambda)
    const int* const ctl = W.st.ctl;

    int64_t bad = -1;
    rpy_status s = first_bad(nb, N, d_precond, &bad, st);
    if (s != RPY_OK) return s;
    if (matvec_prec != RPY_PREC_F64) to_float_kernel<<<vgrid(1), 256, 0, st>>>(d_pos, 0, W.pos32, 0, 3 * N);

    // b_r = [slip_r; -F_r], x = 0, r0 = b
    if (d_slip) axpby_kernel<<<vg, 256, 0, st>>>(1.0, d_slip, 3 * N, 0.0, W.b, ldv, 3 * N);
    else RPY_CUDA_TRY(cudaMemsetAsync(W.b, 0, W.vec_bytes * (size_t)nrhs, st));
    axpby_kernel<<<dim3(64, (unsigned)nrhs), 256, 0, st>>>(-1.0, d_F, 6 * nb, 0.0, W.b + 3 * N, ldv, 6 * nb);
    RPY_CUDA_TRY(cudaMemsetAsync(W.x, 0, W.vec_bytes * (size_t)nrhs, st));
    norm_partial_kernel<<<vg, kVecThreads, 0, st>>>(W.b, ldv, n, W.norm_partial);
    cycle_start_kernel<<<nrhs, 32, 0, st>>>(W.st, W.norm_partial, kVecBlocks, 1);

    // one read-back: the four control words and the scalar state of every right-hand side
    const size_t status_bytes = 64 + sizeof(double) * kScal * (size_t)nrhs;
    alignas(8) unsigned char hbuf[64 + sizeof(double) * kScal * RPY_RIGID_MAX_BATCH];
    const double* hs = reinterpret_cast<const double*>(hbuf + 64);
    auto read_now = [&]() -> cudaError_t {           // after everything enqueued so far
        cudaError_t e = cudaMemcpyAsync(hbuf, W.status, status_bytes, cudaMemcpyDeviceToHost, st);
        return e != cudaSuccess ? e : cudaStreamSynchronize(st);
    };
    // the snapshot the device left at the end of step j (slot j & 1): read after what had been enqueued when
    // mark() was called; step j+1, enqueued in between, writes the other slot
    alignas(8) unsigned char hsnap[kSnapBytes];
    const int* snap_i = reinterpret_cast<const int*>(hsnap);
    const double* snap_res = reinterpret_cast<const double*>(hsnap + 16);
    const size_t snap_bytes = 16 + sizeof(double) * (size_t)nrhs;
    auto mark = [&]() -> cudaError_t { return side ? cudaEventRecord(side_ev, st) : cudaSuccess; };
    auto read_marked = [&](int j) -> cudaError_t {
        const unsigned char* src = W.st.snap + (size_t)(j & 1) * kSnapBytes;
        if (!side) {
            cudaError_t e = cudaMemcpyAsync(hsnap, src, snap_bytes, cudaMemcpyDeviceToHost, st);
            return e != cudaSuccess ? e : cudaStreamSynchronize(st);
        }
        cudaError_t e = cudaStreamWaitEvent(side, side_ev, 0);
        if (e != cudaSuccess) return e;
        e = cudaMemcpyAsync(hsnap, src, snap_bytes, cudaMemcpyDeviceToHost, side);
        return e != cudaSuccess ? e : cudaStreamSynchronize(side);
    };
    RPY_CUDA_TRY(read_now());
    double bnorm[RPY_RIGID_MAX_BATCH], rel[RPY_RIGID_MAX_BATCH];
    bool any = false;
    for (int r = 0; r < nrhs; ++r) {
        bnorm[r] = hs[r * kScal + 3];
        if (!isfinite(bnorm[r])) return RPY_ERR_ARG;
        rel[r] = bnorm[r] > 0.0 ? 1.0 : 0.0;
        any = any || bnorm[r] > 0.0;
        if (h_history) h_history[(size_t)r * (max_iter + 1)] = rel[r];
    }
    auto all_le = [&](const double* v, double t) { for (int r = 0; r < nrhs; ++r) if (v[r] > t) return false; return true; };

    StepEnd end;
    end.enabled = 1; end.j = 0; end.max_iter = max_iter; end.mixed = mixed ? 1 : 0; end.tol = tol;
    end.inner_reduction = kInnerReduction; end.inner_tol_factor = kInnerTolFactor; end.f32_bound = kF32ProductBound;
    StepEnd no_end = end; no_end.enabled = 0;

    // Arnoldi step j of the current cycle; `src` is what v_j is a multiple of (the residual for j = 0, else w)
    auto enqueue_step = [&](int j, const double* src) -> rpy_status {
        double* vj = W.V + (int64_t)j * nrhs * ldv;
        rpy_status e = precond_apply(N, nb, d_precond, src, W.z, ldv, nrhs, st, lam32_in_cycle, W.st.scal, vj, ctl);
        if (e != RPY_OK) return e;
        e = saddle(wall, inner_prec, N, nb, d_pos, d_q, d_offsets, a, eta, W.z, W.w, ldv, nrhs, W, st,
                   lam32_in_cycle != nullptr, ctl, sh);
        if (e != RPY_OK) return e;
        // classical Gram-Schmidt, twice (as accurate as the modified form; three launches for the two passes)
        StepEnd ej = end; ej.j = j;
        const dim3 vt(kVecThreads);
        RPY_CUDA_TRY(rpy::launch_pdl(dots_kernel, vg, vt, 0, st, (const double*)W.V, ldv, nrhs, j + 1, (const double*)W.w, n, W.partial, pvec, ctl));
        RPY_CUDA_TRY(rpy::launch_pdl(update_kernel, vg, vt, 0, st, (const double*)W.V, ldv, nrhs, j + 1, W.w, n, (const double*)W.partial, pvec,
                                     W.st.hcol, 0, W.norm_partial, W.partial2, W.st, no_end, ctl));
        RPY_CUDA_TRY(rpy::launch_pdl(update_kernel, vg, vt, 0, st, (const double*)W.V, ldv, nrhs, j + 1, W.w, n, (const double*)W.partial2, pvec,
                                     W.st.hcol, 1, W.norm_partial, (double*)nullptr, W.st, ej, ctl));
        return RPY_OK;
    };

    int n_iter = 0;
    const double* rvec = W.b;
    bool done = !any;
    bool certified = false;                                  // mixed: the last cycle ended within tol - margin (no fp64 check)
    double start_rel[RPY_RIGID_MAX_BATCH];                   // true relative residual the current cycle started from
    for (int r = 0; r < nrhs; ++r) start_rel[r] = rel[r];
    while (!done) {
        int k = 0;
        int enq = n_iter;                                    // iterations enqueued so far (those of step j included)
        if ((s = enqueue_step(0, rvec)) != RPY_OK) return s;
        ++enq;
        for (int j = 0;; ++j) {
            RPY_CUDA_TRY(mark());
            const bool more = j + 1 < restart && enq < max_iter;
            if (more) {                                      // one step ahead of the device's decision
                if ((s = enqueue_step(j + 1, W.w)) != RPY_OK) return s;
                ++enq;
            }
            RPY_CUDA_TRY(read_marked(j));
            ++n_iter;
            for (int r = 0; r < nrhs; ++r) {
                rel[r] = bnorm[r] > 0.0 ? snap_res[r] / bnorm[r] : 0.0;
                if (h_history) h_history[(size_t)r * (max_iter + 1) + n_iter] = rel[r];
            }
            k = j + 1;
            if (snap_i[0] != 0) {                            // the device closed the cycle at this step
                if (!mixed) done = true;                     // converged, or max_iter reached
                else if (snap_i[1] != 0) {                   // mixed: converged within the margin of the fp32 products
                    done = certified = true;
                    for (int r = 0; r < nrhs; ++r) rel[r] += kF32ProductBound * start_rel[r];   // reported: an upper bound
                }
                break;
            }
            if (!more) break;                                // restart length reached
        }
        // x += P^-1 (V_k y),  R y = g
        solve_y_kernel<<<nrhs, 32, 0, st>>>(W.st, k);
        combine_kernel<<<vg, 256, 0, st>>>(W.V, ldv, nrhs, k, W.st.yv, restart, W.w, n);
        if ((s = precond_apply(N, nb, d_precond, W.w, W.z, ldv, nrhs, st)) != RPY_OK) return s;
        axpby_kernel<<<vg, 256, 0, st>>>(1.0, W.z, ldv, 1.0, W.x, ldv, n);
        const bool want_true_residual = matvec_prec != RPY_PREC_F64 && !certified;   // the estimates were those of the fp32 operator
        if (done && !want_true_residual) break;
        if (!done && !mixed && n_iter >= max_iter) { done = true; if (!want_true_residual) break; }
        // r = b - A x: the start of the next cycle; with fp32 products inside the cycle it is formed with the fp64
        // product -- the true residual of Eq. (11), which decides convergence (mixed) or is what is reported (fp32)
        const rpy_prec rprec = want_true_residual ? RPY_PREC_F64 : outer_prec;
        if ((s = saddle(wall, rprec, N, nb, d_pos, d_q, d_offsets, a, eta, W.x, W.w, ldv, nrhs, W, st, false, nullptr, sh)) != RPY_OK) return s;
        axpby_kernel<<<vg, 256, 0, st>>>(1.0, W.b, ldv, -1.0, W.w, ldv, n);
        norm_partial_kernel<<<vg, kVecThreads, 0, st>>>(W.w, ldv, n, W.norm_partial);
        cycle_start_kernel<<<nrhs, 32, 0, st>>>(W.st, W.norm_partial, kVecBlocks, 0);
        rvec = W.w;
        if (want_true_residual) {
            RPY_CUDA_TRY(read_now());
            for (int r = 0; r < nrhs; ++r) {
                rel[r] = bnorm[r] > 0.0 ? hs[r * kScal + 0] / bnorm[r] : 0.0;
                if (h_history) h_history[(size_t)r * (max_iter + 1) + n_iter] = rel[r];   // replace the estimate by the true value
                start_rel[r] = rel[r];
            }
            if (done) break;                                 // fp32 solve: reported, not iterated on
            if (all_le(rel, tol) || n_iter >= max_iter) done = true;
        }
    }
    axpby_kernel<<<vg, 256, 0, st>>>(1.0, W.x, ldv, 0.0, d_lambda, 3 * N, 3 * N);
    axpby_kernel<<<dim3(64, (unsigned)nrhs), 256, 0, st>>>(1.0, W.x + 3 * N, ldv, 0.0, d_U, 6 * nb, 6 * nb);
    RPY_CUDA_TRY(cudaGetLastError());
    RPY_CUDA_TRY(cudaStreamSynchronize(st));
    if (h_n_iter) *h_n_iter = n_iter;
    if (h_rel_resid) for (int r = 0; r < nrhs; ++r) h_rel_resid[r] = rel[r];
    return RPY_OK;
}

rpy_status solve_checked(int wall, rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies, int n_rhs,
                         const double* d_pos, const double* d_q, const int64_t* d_offsets,
                         const double* d_F, const double* d_slip, double a, double eta,
                         const void* d_precond, double tol, int restart, int max_iter,
                         double* d_lambda, double* d_U, double* h_history, int* h_n_iter, double* h_rel_resid,
                         void* d_workspace, size_t workspace_bytes, void* cuda_stream, const rpy_rigid_solve_ext* ext)
{
    if (matvec_prec != RPY_PREC_F64 && matvec_prec != RPY_PREC_F32_ACC64 && matvec_prec != kPrecMixed) return RPY_ERR_ARG;
    if (check_bodies(n_blobs, n_bodies) != RPY_OK || n_bodies < 1 || n_rhs < 1 || n_rhs > RPY_RIGID_MAX_BATCH) return RPY_ERR_ARG;
    if (!finite_pos(a) || !finite_pos(eta) || !(tol >= 0.0) || restart < 1 || restart > RPY_RIGID_MAX_RESTART || max_iter < 1)
        return RPY_ERR_ARG;
    if (!d_pos || !d_q || !d_offsets || !d_F || !d_precond || !d_lambda || !d_U || !d_workspace) return RPY_ERR_NULL;
    return solve_batch(wall, matvec_prec, n_blobs, n_bodies, n_rhs, d_pos, d_q, d_offsets, d_F, d_slip, a, eta, d_precond,
                       tol, restart, max_iter, d_lambda, d_U, h_history, h_n_iter, h_rel_resid, d_workspace,
                       workspace_bytes, static_cast<cudaStream_t>(cuda_stream), ext);
}

}  // namespace

extern "C" {

rpy_status rpy_rigid_mobility_solve(int wall, rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies,
                                    const double* d_pos, const double* d_q, const int64_t* d_offsets,
                                    const double* d_F, const double* d_slip, double a, double eta,
                                    const void* d_precond, double tol, int restart, int max_iter,
                                    double* d_lambda, double* d_U,
                                    double* h_history, int* h_n_iter, double* h_rel_resid,
                                    void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                                    const rpy_rigid_solve_ext* ext)
{
    return solve_checked(wall, matvec_prec, n_blobs, n_bodies, 1, d_pos, d_q, d_offsets, d_F, d_slip, a, eta, d_precond,
                         tol, restart, max_iter, d_lambda, d_U, h_history, h_n_iter, h_rel_resid, d_workspace,
                         workspace_bytes, cuda_stream, ext);
}

rpy_status rpy_rigid_mobility_solve_batch(int wall, rpy_prec matvec_prec, int64_t n_blobs, int64_t n_bodies, int n_rhs,
                                          const double* d_pos, const double* d_q, const int64_t* d_offsets,
                                          const double* d_F, const double* d_slip, double a, double eta,
                                          const void* d_precond, double tol, int restart, int max_iter,
                                          double* d_lambda, double* d_U,
                                          double* h_history, int* h_n_iter, double* h_rel_resid,
                                          void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                                          const rpy_rigid_solve_ext* ext)
{
    return solve_checked(wall, matvec_prec, n_blobs, n_bodies, n_rhs, d_pos, d_q, d_offsets, d_F, d_slip, a, eta, d_precond,
                         tol, restart, max_iter, d_lambda, d_U, h_history, h_n_iter, h_rel_resid, d_workspace,
                         workspace_bytes, cuda_stream, ext);
}

}  // extern "C"
