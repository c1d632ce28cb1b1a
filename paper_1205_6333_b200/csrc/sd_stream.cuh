// sd_stream.cuh -- the O(N) streaming kernels around the pair kernel (HBM-bound):
//   pack      : caller's pos/force [N][4]  ->  packed records {r | c1 F} (+ pad records); the
//               1/r coefficient c1 = mu0 3a/4 is folded into the force lane (sd_common.cuh)
//   finalize  : sum the segment partials of every row, add the self term mu0 F_i (Eq. 7a,
//               PAPER.md:70-73), write vel, and -- fused -- apply the integrator update
//               (Euler r <- r + dt v; midpoint half / full stage) including the
//               refresh of the packed records for the next product.
// In the fp32 modes positions are carried as (hi, lo) float pairs (double-single, PAPER.md:253,
// :263): the update is formed in fp64 from hi + lo + dt v and split again.
#pragma once
#include "sd_common.cuh"
#include "sd_pairs_f32.cuh"
#include "sd_pairs_f64.cuh"

namespace sd {

enum { FIN_VEL = 0, FIN_EULER = 1, FIN_HALF = 2, FIN_FULL = 3 };
enum { PACK_POS = 1, PACK_FORCE = 2, PACK_GRAVITY = 4 };

// T4 = float4 / double4
template <typename T4>
struct Vec4;
template <>
struct Vec4<float4> {
    typedef float S;
    static __device__ __forceinline__ float4 make(float x, float y, float z, float w) {
        return make_float4(x, y, z, w);
    }
};
template <>
struct Vec4<double4> {
    typedef double S;
    static __device__ __forceinline__ double4 make(double x, double y, double z, double w) {
        return make_double4(x, y, z, w);
    }
};

template <typename T4>
__global__ void __launch_bounds__(256)
pack_kernel(const T4* __restrict__ pos, const T4* __restrict__ force, T4* __restrict__ rec,
            const int what, const double gx, const double gy, const double gz, const double c1,
            const int N, const int Nrec) {
    typedef typename Vec4<T4>::S S;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Nrec) return;
    if (i < N) {
        if (what & PACK_POS) {
            const T4 p = pos[i];
            rec[2 * static_cast<size_t>(i)] = Vec4<T4>::make(p.x, p.y, p.z, S(0));
        }
        if (what & PACK_FORCE) {
            const T4 f = force[i];
            const S k = S(c1);
            rec[2 * static_cast<size_t>(i) + 1] = Vec4<T4>::make(k * f.x, k * f.y, k * f.z, S(0));
        } else if (what & PACK_GRAVITY) {
            rec[2 * static_cast<size_t>(i) + 1] = Vec4<T4>::make(S(c1 * gx), S(c1 * gy), S(c1 * gz), S(0));
        }
    } else {
        const S pp = S(SD_PAD_POS);
        rec[2 * static_cast<size_t>(i)] = Vec4<T4>::make(pp, pp, pp, S(0));
        rec[2 * static_cast<size_t>(i) + 1] = Vec4<T4>::make(S(0), S(0), S(0), S(0));
    }
}

// uniform force written out per particle (sd_step with gravity on the paths that read a force array)
template <typename T4>
__global__ void __launch_bounds__(256)
fill4_kernel(T4* __restrict__ out, const double x, const double y, const double z, const int n) {
    typedef typename Vec4<T4>::S S;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = Vec4<T4>::make(S(x), S(y), S(z), S(0));
}

constexpr int kFinThreads = 128;
constexpr int kFinBatch = 8;

// fp32 modes.  part: [slot][Nrec][2] float4 (hi, lo), value = hi - lo.
template <int MODE>
__global__ void __launch_bounds__(kFinThreads)
finalize_f32_kernel(const float4* __restrict__ part, const int* __restrict__ blk_nslots,
                    float4* __restrict__ rec, float4* __restrict__ vel, float4* __restrict__ pos,
                    float4* __restrict__ pos_lo, float4* __restrict__ pos_half, const double dt,
                    const double mu0r, const int N, const int IB, const long long slot_stride,
                    const int pos_comp, const int tensor, const float clampv, const float k2) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int nslots = blk_nslots[i / IB];
    const float4 f = rec[2 * static_cast<size_t>(i) + 1];
    // self term mu0 F_i = (mu0 / c1) (c1 F_i), minus the clamped self-pair term A_c F'_i that the
    // pair kernel's careful pass left in the partial sums (sd_pairs_f32.cuh)
    const double sc = mu0r - static_cast<double>(self_clamped_coef(tensor, clampv, k2));
    double vx = sc * static_cast<double>(f.x);
    double vy = sc * static_cast<double>(f.y);
    double vz = sc * static_cast<double>(f.z);
    // slots in batches of kFinBatch: the loads of a batch are in flight together (a small-N
    // product has up to T slots per row and this kernel is pure latency); the sum keeps slot order
    for (int s0 = 0; s0 < nslots; s0 += kFinBatch) {
        float4 hi[kFinBatch], lo[kFinBatch];
#pragma unroll
        for (int q = 0; q < kFinBatch; ++q) {
            if (s0 + q < nslots) {
                const float4* p = part + (static_cast<size_t>(s0 + q) * slot_stride + i) * 2;
                hi[q] = p[0];
                lo[q] = p[1];
            }
        }
#pragma unroll
        for (int q = 0; q < kFinBatch; ++q) {
            if (s0 + q < nslots) {
                vx += static_cast<double>(hi[q].x) - static_cast<double>(lo[q].x);
                vy += static_cast<double>(hi[q].y) - static_cast<double>(lo[q].y);
                vz += static_cast<double>(hi[q].z) - static_cast<double>(lo[q].z);
            }
        }
    }
    vel[i] = make_float4(static_cast<float>(vx), static_cast<float>(vy), static_cast<float>(vz), 0.f);
    if (MODE == FIN_VEL) return;
    const float4 ph = pos[i];
    const float4 pl = pos_comp ? pos_lo[i] : make_float4(0.f, 0.f, 0.f, 0.f);  // 0: plain fp32 positions
    const double h = (MODE == FIN_HALF) ? 0.5 * dt : dt;
    const double X = (static_cast<double>(ph.x) + static_cast<double>(pl.x)) + h * vx;
    const double Y = (static_cast<double>(ph.y) + static_cast<double>(pl.y)) + h * vy;
    const double Z = (static_cast<double>(ph.z) + static_cast<double>(pl.z)) + h * vz;
    const float xh = static_cast<float>(X), yh = static_cast<float>(Y), zh = static_cast<float>(Z);
    rec[2 * static_cast<size_t>(i)] = make_float4(xh, yh, zh, 0.f);
    if (MODE == FIN_HALF) {  // r_h only feeds the second product (and a force callback)
        pos_half[i] = make_float4(xh, yh, zh, 0.f);
        return;
    }
    pos[i] = make_float4(xh, yh, zh, 0.f);
    pos_lo[i] = pos_comp ? make_float4(static_cast<float>(X - static_cast<double>(xh)),
                                       static_cast<float>(Y - static_cast<double>(yh)),
                                       static_cast<float>(Z - static_cast<double>(zh)), 0.f)
                         : make_float4(0.f, 0.f, 0.f, 0.f);
}

// fp64 mode.  part: [slot][Nrec] double4.
template <int MODE>
__global__ void __launch_bounds__(kFinThreads)
finalize_f64_kernel(const double4* __restrict__ part, const int* __restrict__ blk_nslots,
                    double4* __restrict__ rec, double4* __restrict__ vel,
                    double4* __restrict__ pos, double4* __restrict__ pos_half, const double dt,
                    const double mu0r, const int N, const int IB, const long long slot_stride,
                    const int tensor, const double clampv, const double k2) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int nslots = blk_nslots[i / IB];
    const double4 f = rec[2 * static_cast<size_t>(i) + 1];
    const double sc = mu0r - self_clamped_coef_f64(tensor, clampv, k2);  // see finalize_f32_kernel
    double vx = sc * f.x, vy = sc * f.y, vz = sc * f.z;
    for (int s0 = 0; s0 < nslots; s0 += kFinBatch) {
        double4 p[kFinBatch];
#pragma unroll
        for (int q = 0; q < kFinBatch; ++q)
            if (s0 + q < nslots) p[q] = part[static_cast<size_t>(s0 + q) * slot_stride + i];
#pragma unroll
        for (int q = 0; q < kFinBatch; ++q) {
            if (s0 + q < nslots) {
                vx += p[q].x;
                vy += p[q].y;
                vz += p[q].z;
            }
        }
    }
    vel[i] = make_double4(vx, vy, vz, 0.0);
    if (MODE == FIN_VEL) return;
    const double4 p0 = pos[i];
    const double h = (MODE == FIN_HALF) ? 0.5 * dt : dt;
    const double4 pn = make_double4(p0.x + h * vx, p0.y + h * vy, p0.z + h * vz, 0.0);
    rec[2 * static_cast<size_t>(i)] = pn;
    if (MODE == FIN_HALF) {
        pos_half[i] = pn;
        return;
    }
    pos[i] = pn;
}

// FMA-peak probes (roofline calibration): K independent dependent-chains per thread.
__global__ void __launch_bounds__(512)
fma_probe_f32_kernel(float* out, const float a, const float b, const int iters) {
    float x[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) x[q] = threadIdx.x * 1e-3f + q;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int q = 0; q < 8; ++q) x[q] = fmaf(x[q], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += x[q];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(512)
fma_probe_f64_kernel(double* out, const double a, const double b, const int iters) {
    double x[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) x[q] = threadIdx.x * 1e-3 + q;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int q = 0; q < 8; ++q) x[q] = fma(x[q], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += x[q];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace sd
