// sd_small.cuh -- the small-N path (below a few thousand
// particles the device is under-filled and the run time is linear in N).
//
// For small N the all-pairs arithmetic is microseconds; what counts is the number of launches and
// how many SMs get work.  Two kernels, both evaluating every pair with the exact branching body
// (self exclusion, coincident centres, r < 2a branch) -- no fast/slow split is worth it here:
//
//  small_apply_kernel   N <= kSmallApplyMax.  ONE launch per product, straight from the caller's
//      pos/force arrays (no pack, no partial buffer, no finalize).  A warp owns IPW particles i
//      and its 32 lanes split j (lane l takes j = l, l+32, ...); j tiles of 256 records are staged
//      in shared memory by the whole CTA; per-lane Kahan sums are combined by warp shuffles of the
//      3-vector in fp64; lane 0 adds mu0 F_i, writes vel and applies the fused integrator update
//      (Euler needs ping-pong position buffers, the midpoint stages do not).
//      Grid = N / (8 IPW) CTAs, IPW chosen so that every SM gets a CTA as early as possible.
//
//  small_stepper_kernel N <= kStepperMax, constant forces.  ONE launch for n_steps steps: a
//      single CTA keeps the positions in shared memory (fp64 = hi + lo of the fp32 modes), S lanes
//      per particle split j, shuffle reduction, two block barriers per product.  Removes the
//      launch latency (~10 us per 4-launch step) that dominates N = 4 (config 1) and makes the
//      5e7-step stability runs of PAPER.md:253 a matter of seconds.
#pragma once
#include "sd_common.cuh"
#include "sd_pairs_f32.cuh"
#include "sd_stream.cuh"

namespace sd {

constexpr int kSmallApplyMax = 2560;  // above this the tiled packed kernel wins (measured)
constexpr int kStepperMax = 64;   // above this one launch per product is faster (measured)
constexpr int kSmallThreads = 256;
constexpr int kSmallTile = 256;

template <typename S>
struct CoefT {
    S c1, c2, m3c2, mu0, ovA, ovB, four_a2;
    // periodic cube (PAPER.md:115 footnote 1): invL = 0 means free space; see PairCoefT
    S invL, mL, magic;
};

// nearest image of one displacement component, same rule as the tiled kernels (the branch is
// uniform over the grid)
__device__ __forceinline__ float min_image(const float d, const CoefT<float>& k) {
    if (k.invL == 0.0f) return d;
    return __fmaf_rn(__fsub_rn(__fmaf_rn(d, k.invL, k.magic), k.magic), k.mL, d);
}
__device__ __forceinline__ double min_image(const double d, const CoefT<double>& k) {
    if (k.invL == 0.0) return d;
    return fma(__dsub_rn(fma(d, k.invL, k.magic), k.magic), k.mL, d);
}

__device__ __forceinline__ float inv_sqrt_exact(float r2) {
    float y = rsq_approx(r2);
    // one Newton step: the small path is not throughput-bound, take the extra bits
    const float e = fmaf(-r2 * y, y, 1.0f);
    return fmaf(0.5f * y, e, y);
}
__device__ __forceinline__ double inv_sqrt_exact(double r2) { return 1.0 / sqrt(r2); }

// One exact pair term added to (px, py, pz); `self` pairs are skipped.
template <typename S, int TENSOR>
__device__ __forceinline__ void pair_term(const S xi, const S yi, const S zi, const bool self,
                                          const S xj, const S yj, const S zj, const S fx,
                                          const S fy, const S fz, const CoefT<S>& k, S& px, S& py,
                                          S& pz) {
    if (self) return;
    const S dx = min_image(xi - xj, k), dy = min_image(yi - yj, k), dz = min_image(zi - zj, k);
    const S r2 = dx * dx + dy * dy + dz * dz;
    if (r2 == S(0)) {
        if (TENSOR == TENSOR_RPY) {
            px += k.mu0 * fx;
            py += k.mu0 * fy;
            pz += k.mu0 * fz;
        }
        return;
    }
    const S inv = inv_sqrt_exact(r2);
    const S dF = dx * fx + dy * fy + dz * fz;
    S A, B;
    if (TENSOR == TENSOR_RPY) {
        if (r2 < k.four_a2) {
            const S r = r2 * inv;
            A = k.mu0 + k.ovA * r;
            B = k.ovB * inv;
        } else {
            const S inv2 = inv * inv;
            A = (k.c1 + k.c2 * inv2) * inv;
            B = (k.c1 + k.m3c2 * inv2) * inv2 * inv;
        }
    } else {
        A = k.c1 * inv;
        B = A * inv * inv;
    }
    const S Bd = B * dF;
    px += A * fx + Bd * dx;
    py += A * fy + Bd * dy;
    pz += A * fz + Bd * dz;
}

// Kahan (KAHAN = true) or plain running sum of 3-vectors.
template <typename S, bool KAHAN>
struct Acc3 {
    S sx = S(0), sy = S(0), sz = S(0), cx = S(0), cy = S(0), cz = S(0);
    __device__ __forceinline__ void add(const S tx, const S ty, const S tz) {
        if (KAHAN) {
            S y = tx - cx, t = sx + y;
            cx = (t - sx) - y;
            sx = t;
            y = ty - cy, t = sy + y;
            cy = (t - sy) - y;
            sy = t;
            y = tz - cz, t = sz + y;
            cz = (t - sz) - y;
            sz = t;
        } else {
            sx += tx;
            sy += ty;
            sz += tz;
        }
    }
    __device__ __forceinline__ void value(double& x, double& y, double& z) const {
        x = static_cast<double>(sx) - static_cast<double>(cx);
        y = static_cast<double>(sy) - static_cast<double>(cy);
        z = static_cast<double>(sz) - static_cast<double>(cz);
    }
};

template <int WIDTH>
__device__ __forceinline__ double lanes_sum(double v) {
#pragma unroll
    for (int o = WIDTH / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o, WIDTH);
    return v;
}

template <int WIDTH>
__device__ __forceinline__ float lanes_sum_f32(float v) {
#pragma unroll
    for (int o = WIDTH / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o, WIDTH);
    return v;
}

// Cross-lane sum of the per-lane partial sums + self term mu0 F_i.  Compensated modes and fp64
// combine in fp64; SD_PREC_F32_PLAIN stays in fp32 throughout, so that "single-precision
// accumulation" means what it says even when a lane holds a single term.
template <typename S, bool KAHAN, int WIDTH>
__device__ __forceinline__ void combine_lanes(const Acc3<S, KAHAN>& acc, const S mu0, const S fx,
                                              const S fy, const S fz, double& vx, double& vy,
                                              double& vz) {
    acc.value(vx, vy, vz);
    if (!KAHAN && sizeof(S) == 4) {
        const float m = static_cast<float>(mu0);
        vx = fmaf(m, static_cast<float>(fx), lanes_sum_f32<WIDTH>(static_cast<float>(vx)));
        vy = fmaf(m, static_cast<float>(fy), lanes_sum_f32<WIDTH>(static_cast<float>(vy)));
        vz = fmaf(m, static_cast<float>(fz), lanes_sum_f32<WIDTH>(static_cast<float>(vz)));
    } else {
        vx = lanes_sum<WIDTH>(vx) + static_cast<double>(mu0) * static_cast<double>(fx);
        vy = lanes_sum<WIDTH>(vy) + static_cast<double>(mu0) * static_cast<double>(fy);
        vz = lanes_sum<WIDTH>(vz) + static_cast<double>(mu0) * static_cast<double>(fz);
    }
}

// ---- one product per launch -----------------------------------------------------------------
// posx: positions the distances are taken from; force: per-particle forces or NULL (uniform g).
// MODE (sd_stream.cuh, run-time): FIN_VEL writes vel only; otherwise pos_base (+ pos_lo) + h v
// -> pos_out.
template <typename T4, int TENSOR, bool KAHAN, int IPW>
__global__ void __launch_bounds__(kSmallThreads)
small_apply_kernel(const T4* __restrict__ posx, const T4* __restrict__ force, const double gx,
                   const double gy, const double gz, T4* __restrict__ vel,
                   const T4* __restrict__ pos_base, T4* __restrict__ pos_lo,
                   T4* __restrict__ pos_out, const double dt, const int MODE,
                   const CoefT<typename Vec4<T4>::S> k, const int N, const int pos_comp) {
    typedef typename Vec4<T4>::S S;
    __shared__ T4 sp[kSmallTile];
    __shared__ T4 sf[kSmallTile];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i0 = (blockIdx.x * (kSmallThreads / 32) + warp) * IPW;
    S xi[IPW], yi[IPW], zi[IPW];
    Acc3<S, KAHAN> acc[IPW];
#pragma unroll
    for (int m = 0; m < IPW; ++m) {
        const int i = min(i0 + m, N - 1);
        const T4 p = posx[i];
        xi[m] = p.x;
        yi[m] = p.y;
        zi[m] = p.z;
    }
    for (int j0 = 0; j0 < N; j0 += kSmallTile) {
        const int j = j0 + tid;
        if (j < N) {
            sp[tid] = posx[j];
            sf[tid] = force ? force[j] : Vec4<T4>::make(S(gx), S(gy), S(gz), S(0));
        }
        __syncthreads();
        const int nj = min(kSmallTile, N - j0);
        for (int jj = lane; jj < nj; jj += 32) {
            const T4 pj = sp[jj];
            const T4 fj = sf[jj];
#pragma unroll
            for (int m = 0; m < IPW; ++m) {
                S tx = S(0), ty = S(0), tz = S(0);
                pair_term<S, TENSOR>(xi[m], yi[m], zi[m], (j0 + jj) == (i0 + m), pj.x, pj.y, pj.z,
                                     fj.x, fj.y, fj.z, k, tx, ty, tz);
                acc[m].add(tx, ty, tz);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int m = 0; m < IPW; ++m) {
        const int i = i0 + m;
        S sfx = S(gx), sfy = S(gy), sfz = S(gz);  // F_i of the self term
        if (force) {
            const T4 f = force[min(i, N - 1)];
            sfx = f.x, sfy = f.y, sfz = f.z;
        }
        double vx, vy, vz;
        combine_lanes<S, KAHAN, 32>(acc[m], k.mu0, sfx, sfy, sfz, vx, vy, vz);
        if (lane == 0 && i < N) {
            vel[i] = Vec4<T4>::make(S(vx), S(vy), S(vz), S(0));
            if (MODE != FIN_VEL) {
                const T4 ph = pos_base[i];
                double X = ph.x, Y = ph.y, Z = ph.z;
                if (sizeof(S) == 4 && pos_comp) {
                    const T4 pl = pos_lo[i];
                    X += pl.x, Y += pl.y, Z += pl.z;
                }
                const double h = (MODE == FIN_HALF) ? 0.5 * dt : dt;
                X += h * vx, Y += h * vy, Z += h * vz;
                const S xh = S(X), yh = S(Y), zh = S(Z);
                pos_out[i] = Vec4<T4>::make(xh, yh, zh, S(0));
                if (MODE != FIN_HALF && sizeof(S) == 4)  // pos_comp = 0: plain fp32 positions
                    pos_lo[i] = pos_comp ? Vec4<T4>::make(S(X - static_cast<double>(xh)),
                                                          S(Y - static_cast<double>(yh)),
                                                          S(Z - static_cast<double>(zh)), S(0))
                                         : Vec4<T4>::make(S(0), S(0), S(0), S(0));
            }
        }
    }
}

// ---- one product per launch, fp32, packed arithmetic -------------------------------------------
// Same mapping as small_apply_kernel (a warp owns two particles, its lanes split j, tiles staged
// by the CTA, shuffle reduction, fused integrator update), but the pair arithmetic is the packed
// "careful" body of the tiled kernel (sd_pairs_f32.cuh): the two particles of a warp are the two
// halves of f32x2 registers, r^2 is clamped from below so that every pair -- self pair included --
// adds a finite term, and the pairs below the clamp are put right one by one (clamped term out,
// exact term in).  ~30 instead of ~110 instructions per two pairs.  Works in the folded units of
// the tiled kernels on the caller's raw forces: the sum is multiplied by c1 = mu0 3a/4 at the end.
// Compensation: plain adds over the (at most 4) terms a lane takes from a 128-record tile, Kahan
// merge per 128 j.  CTAs of 128 threads = 8 particles: N / 8 CTAs; the CTA keeps all N records in
// shared memory.
constexpr int kPackedThreads = 128;
// Measured window (products replayed from a CUDA graph, us per product, free space): against the scalar
// warp-per-particle kernel N = 256 3.04 (3.06), 384 3.63 (4.09), 512 3.51 (4.76), 768 4.73 (5.92 before the
// unrolling below); against the warp-split kernel (sd_pairs_f32w.cuh) with CTAs of 512 threads N = 2560 16.1
// (19.9), 3000 17.8 (22.2), 4096 23.0 (28.0), 4736 26.4 (35.6).  Above 4736 the CTAs no longer fit one per SM
// (32 N bytes of shared memory each); in the periodic box the warp-split kernel wins from 2304 on (N = 4000:
// 29.6 against 28.1 us per Euler step with the packed kernel forced, but 20.7 against 21.6 at N = 2916: no window worth a second threshold).  Round 1 (128-record chunks, rolled loop): N = 1024 6.5, 2048 12.7 us.
constexpr int kPackedMinN = 256;
constexpr int kPackedMaxN = 4736;      // 148 SMs x 32 particles: one CTA of 512 threads per SM
constexpr int kPackedMaxNBox = 2304;   // default limit in the periodic box (29 instead of 20 packed instructions per step: the warp-split kernel's 8 particles per lane win from here on)
constexpr int kPackedWideMinN = 2305;  // above: CTAs of 512 threads (32 particles), 32 N bytes of shared memory each
__host__ __device__ constexpr int packed_threads(int n) { return n >= kPackedWideMinN ? 512 : kPackedThreads; }
constexpr int kPackedTile = 256;

template <int TENSOR, bool KAHAN, bool PBC, int THREADS = kPackedThreads>
__global__ void __launch_bounds__(THREADS)
small_apply_packed_kernel(const float4* __restrict__ posx, const float4* __restrict__ force,
                          const double gx, const double gy, const double gz,
                          float4* __restrict__ vel, const float4* __restrict__ pos_base,
                          float4* __restrict__ pos_lo, float4* __restrict__ pos_out, const double dt,
                          const int MODE, const PairCoef k, const double c1, const double mu0,
                          const int N, const int pos_comp) {
    // all N records (positions, then forces) in dynamic shared memory: 32 N bytes <= 80 KiB, one
    // barrier per product instead of two per tile (at these sizes the kernel is latency, not
    // arithmetic: 8 serial tile hand-overs cost more than the pairs)
    extern __shared__ float4 s_all[];
    float4* sp = s_all;
    float4* sf = s_all + N;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i0 = (blockIdx.x * (THREADS / 32) + warp) * 2;
    const int ia = min(i0, N - 1), ib = min(i0 + 1, N - 1);
    // (unrolled: the loads of four iterations are in flight together; the loop is pure L2 latency)
#pragma unroll 4
    for (int j = tid; j < N; j += THREADS) {
        sp[j] = posx[j];
        sf[j] = force ? force[j] : make_float4(float(gx), float(gy), float(gz), 0.f);
    }
    __syncthreads();
    const float4 pa = sp[ia], pb = sp[ib];
    const f32x2 zero = bc2(0.f);
    f32x2 xi[1] = {add2(pk2(pa.x, pb.x), zero)}, yi[1] = {add2(pk2(pa.y, pb.y), zero)},
          zi[1] = {add2(pk2(pa.z, pb.z), zero)};
    f32x2 sx = zero, sy = zero, sz = zero, cx = zero, cy = zero, cz = zero;
    // 256-record chunks with 128 threads (eight j per lane in flight); 128-record chunks with 512 threads, where
    // the 128-register cap would otherwise spill (24 ... 48 B of stack: N = 4096 23.9 -> 23.0 us without)
    constexpr int kTile = (THREADS > kPackedThreads) ? 128 : kPackedTile;
    for (int j0 = 0; j0 < N; j0 += kTile) {   // compensation chunk: kTile / 32 terms per lane
        const int nj = min(j0 + kTile, N);
        f32x2 px[1] = {zero}, py[1] = {zero}, pz[1] = {zero};
        // the (at most four) j of a lane: first the clamped packed body of all of them as straight-line code, so
        // that their address, distance, MUFU and coefficient stages overlap (one warp per scheduler: nothing else
        // hides those latencies; N = 1024: 6.5 -> 5.9 us per product with the four bodies unrolled), then the rare
        // pairs below the clamp are put right one by one
        constexpr int kPerLane = kTile / 32;
        float r2q[kPerLane][2];
        auto fast_j = [&](const int q, const int j) {
            float mn = 0.f;
            pair_fast_staged<1, TENSOR, PBC, true>(xi, yi, zi, sp[j], sf[j], k, px, py, pz, mn, r2q[q]);
        };
        auto fix_j = [&](const int q, const int j) {
            if (fminf(r2q[q][0], r2q[q][1]) < k.clampv) {
                const float4 pj = sp[j];
                const float4 fj = sf[j];
                float ax = lo2(px[0]), ay = lo2(py[0]), az = lo2(pz[0]);
                float bx = hi2(px[0]), by = hi2(py[0]), bz = hi2(pz[0]);
                if (r2q[q][0] < k.clampv) {
                    pair_clamped_sub<TENSOR, PBC>(pa.x, pa.y, pa.z, pj, fj, k, ax, ay, az);
                    pair_exact<TENSOR, PBC>(pa.x, pa.y, pa.z, j == ia, pj, fj, k, ax, ay, az);
                }
                if (r2q[q][1] < k.clampv) {
                    pair_clamped_sub<TENSOR, PBC>(pb.x, pb.y, pb.z, pj, fj, k, bx, by, bz);
                    pair_exact<TENSOR, PBC>(pb.x, pb.y, pb.z, j == ib, pj, fj, k, bx, by, bz);
                }
                px[0] = pk2(ax, bx);
                py[0] = pk2(ay, by);
                pz[0] = pk2(az, bz);
            }
        };
        if (nj - j0 == kTile) {
#pragma unroll
            for (int q = 0; q < kPerLane; ++q) fast_j(q, j0 + lane + 32 * q);
#pragma unroll
            for (int q = 0; q < kPerLane; ++q) fix_j(q, j0 + lane + 32 * q);
        } else {
            for (int j = j0 + lane; j < nj; j += 32) {
                fast_j(0, j);
                fix_j(0, j);
            }
        }
        if (KAHAN) {
            kahan_merge2(sx, cx, px[0]);
            kahan_merge2(sy, cy, py[0]);
            kahan_merge2(sz, cz, pz[0]);
        } else {
            sx = add2(sx, px[0]);
            sy = add2(sy, py[0]);
            sz = add2(sz, pz[0]);
        }
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int i = i0 + h;
        const float hx = h ? hi2(sx) : lo2(sx), hy = h ? hi2(sy) : lo2(sy), hz = h ? hi2(sz) : lo2(sz);
        const float lx = h ? hi2(cx) : lo2(cx), ly = h ? hi2(cy) : lo2(cy), lz = h ? hi2(cz) : lo2(cz);
        float4 fi = make_float4(float(gx), float(gy), float(gz), 0.f);
        if (force) fi = sf[min(i, N - 1)];
        double vx, vy, vz;
        if (KAHAN) {
            vx = lanes_sum<32>(double(hx) - double(lx)) * c1 + mu0 * double(fi.x);
            vy = lanes_sum<32>(double(hy) - double(ly)) * c1 + mu0 * double(fi.y);
            vz = lanes_sum<32>(double(hz) - double(lz)) * c1 + mu0 * double(fi.z);
        } else {  // SD_PREC_F32_PLAIN: fp32 end to end
            const float cf = float(c1), mf = float(mu0);
            vx = fmaf(mf, fi.x, cf * lanes_sum_f32<32>(hx));
            vy = fmaf(mf, fi.y, cf * lanes_sum_f32<32>(hy));
            vz = fmaf(mf, fi.z, cf * lanes_sum_f32<32>(hz));
        }
        if (lane == 0 && i < N) {
            vel[i] = make_float4(float(vx), float(vy), float(vz), 0.f);
            if (MODE != FIN_VEL) {
                const float4 ph = pos_base[i];
                double X = ph.x, Y = ph.y, Z = ph.z;
                if (pos_comp) {
                    const float4 pl = pos_lo[i];
                    X += pl.x, Y += pl.y, Z += pl.z;
                }
                const double hh = (MODE == FIN_HALF) ? 0.5 * dt : dt;
                X += hh * vx, Y += hh * vy, Z += hh * vz;
                const float xh = float(X), yh = float(Y), zh = float(Z);
                pos_out[i] = make_float4(xh, yh, zh, 0.f);
                if (MODE != FIN_HALF)
                    pos_lo[i] = pos_comp ? make_float4(float(X - double(xh)), float(Y - double(yh)),
                                                       float(Z - double(zh)), 0.f)
                                         : make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
    }
}

// ---- all steps in one launch ------------------------------------------------------------------
// One CTA of N * SUB threads (SUB lanes per particle, SUB | 32).  Positions live in shared memory
// as doubles (= hi + lo of the fp32 modes); the pair arithmetic runs in S on S-rounded positions,
// exactly like the large-N path.  integrator: 0 Euler, 1 midpoint.
template <typename T4, int TENSOR, bool KAHAN, int SUB>
__global__ void __launch_bounds__(1024)
small_stepper_kernel(T4* __restrict__ pos, T4* __restrict__ pos_lo, const T4* __restrict__ force,
                     const double gx, const double gy, const double gz, T4* __restrict__ vel,
                     const double dt, const long long n_steps, const int integrator,
                     const CoefT<typename Vec4<T4>::S> k, const int N, const int pos_comp) {
    typedef typename Vec4<T4>::S S;
    __shared__ double P[kStepperMax][3];   // current positions r_n
    __shared__ S X[kStepperMax][3];        // positions the distances are taken from (S-rounded)
    __shared__ S F[kStepperMax][3];
    const int tid = threadIdx.x;
    const int i = tid / SUB, sub = tid % SUB;
    const bool owner = (sub == 0) && (i < N);
    if (owner) {
        const T4 p = pos[i];
        double x = p.x, y = p.y, z = p.z;
        if (sizeof(S) == 4 && pos_comp) {
            const T4 l = pos_lo[i];
            x += l.x, y += l.y, z += l.z;
        }
        P[i][0] = x, P[i][1] = y, P[i][2] = z;
        X[i][0] = S(x), X[i][1] = S(y), X[i][2] = S(z);
        if (force) {
            const T4 f = force[i];
            F[i][0] = f.x, F[i][1] = f.y, F[i][2] = f.z;
        } else {
            F[i][0] = S(gx), F[i][1] = S(gy), F[i][2] = S(gz);
        }
    }
    __syncthreads();
    double vx = 0.0, vy = 0.0, vz = 0.0;
    const int n_products = (integrator == 1) ? 2 : 1;
    for (long long step = 0; step < n_steps; ++step) {
        for (int stage = 0; stage < n_products; ++stage) {
            Acc3<S, KAHAN> acc;
            if (i < N) {
                const S xi = X[i][0], yi = X[i][1], zi = X[i][2];
                for (int j = sub; j < N; j += SUB) {
                    S tx = S(0), ty = S(0), tz = S(0);
                    pair_term<S, TENSOR>(xi, yi, zi, j == i, X[j][0], X[j][1], X[j][2], F[j][0],
                                         F[j][1], F[j][2], k, tx, ty, tz);
                    acc.add(tx, ty, tz);
                }
            }
            {
                const int ii = (i < N) ? i : 0;
                combine_lanes<S, KAHAN, SUB>(acc, k.mu0, F[ii][0], F[ii][1], F[ii][2], vx, vy, vz);
            }
            __syncthreads();  // every lane has read X
            if (owner) {
                const bool half = (n_products == 2) && (stage == 0);
                const double h = half ? 0.5 * dt : dt;
                const double x = P[i][0] + h * vx, y = P[i][1] + h * vy, z = P[i][2] + h * vz;
                X[i][0] = S(x), X[i][1] = S(y), X[i][2] = S(z);
                if (!half) {  // pos_comp = 0: the position is kept in S only ("single")
                    P[i][0] = pos_comp ? x : static_cast<double>(X[i][0]);
                    P[i][1] = pos_comp ? y : static_cast<double>(X[i][1]);
                    P[i][2] = pos_comp ? z : static_cast<double>(X[i][2]);
                }
            }
            __syncthreads();
        }
    }
    if (owner) {
        const S xh = S(P[i][0]), yh = S(P[i][1]), zh = S(P[i][2]);
        pos[i] = Vec4<T4>::make(xh, yh, zh, S(0));
        if (sizeof(S) == 4)
            pos_lo[i] = Vec4<T4>::make(S(P[i][0] - static_cast<double>(xh)),
                                       S(P[i][1] - static_cast<double>(yh)),
                                       S(P[i][2] - static_cast<double>(zh)), S(0));
        vel[i] = Vec4<T4>::make(S(vx), S(vy), S(vz), S(0));
    }
}

}  // namespace sd
