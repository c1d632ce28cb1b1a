// sd_pairs_f64.cuh -- all-pairs mobility kernel, everything in fp64 (SD_PREC_F64).
//
// Same decomposition, staging ring and chunk-level slow path as the fp32 kernel
// (sd_pairs_f32.cuh); differences:
//  * 64-byte records {x, y, z, 0 | Fx, Fy, Fz, 0} of doubles, 64 j per 4 KiB tile;
//  * no packed arithmetic (there is no DFMA2); one thread owns I particles (4 at large N with
//    one CTA per SM, 2 with two CTAs per SM below: halves the LDS.128 per pair);
//  * 1/r: MUFU.RSQ on the fp32-rounded r^2 as a 22-bit seed, then one Newton step in fp64
//    (relative error ~2e-7 -> <= 8.6e-14, see rsqrt_nr2); no fp64 division or sqrt in the loop;
//  * fp64 sums need no compensation (measured 2e-13 vs the oracle's long-double rows at
//    N = 65536); min r^2 is tracked on the fp32 copy of r^2 that the seed needs anyway.
#pragma once
#include "sd_common.cuh"
#include "sd_pairs_f32.cuh"

namespace sd {

constexpr int kTJ64 = 64;  // j records per tile (4 KiB)
// 128-record tiles (8 KiB) for 4 particles per thread at N >= kRepairMaxN: half the tile hand-overs (see kTJLarge in
// sd_pairs_f32.cuh); measured 0.5436 -> 0.5465 of the DFMA roofline at N = 1 M, 0.5426 -> 0.5455 at 262 144.
constexpr int kTJ64Large = 128;

// y0 = MUFU.RSQ(float(r2)) has relative error d0 <= 2^-22.4 + 2^-24 (MUFU + the rounding of r2 to
// float) ~ 2.4e-7.  With e = 1 - r2 y0^2 ~ -2 d0 (a cancellation: fp64), one Newton step
//   y = y0 + y0 e / 2
// leaves a relative error of 3/8 e^2 <= 8.6e-14 in 1/r (always too small), i.e. <= 2.6e-13 in the
// 1/r^3 terms: 40x below the 1e-11 tolerance of this path, in 4 fp64 instructions.  The kernel is
// bound by the FP64 pipe (80 % active, 2 cycles per warp instruction), so the count matters:
//   Newton (shipped)                      25 fp64 instructions per pair   5.985e11 pairs/s at N = 1 M
//   Halley, y0 e (1/2 + 3e/8)  (measured in round 1, removed)   26, error ~1e-21    5.736e11
//   Halley with the correction in fp32 (measured in round 1, removed)  24 + 2 F2F   5.549e11
__device__ __forceinline__ double rsqrt_nr2(const double r2, const float r2f) {
    const float yf = rsq_approx(r2f);
    const double y = static_cast<double>(yf);
    const double e = fma(-r2, y * y, 1.0);
    return fma(y * e, 0.5, y);
}

// fp64 counterpart of self_clamped_coef (sd_pairs_f32.cuh): what pair_fast_f64<CLAMP> multiplies
// F'_i with for the self pair.
__device__ __forceinline__ double self_clamped_coef_f64(const int tensor, const double clampv, const double k2) {
    const double inv = rsqrt_nr2(clampv, static_cast<float>(clampv));
    const double inv2 = inv * inv;
    const double inv3 = inv2 * inv;
    return tensor == TENSOR_RPY ? fma(k2, inv3, inv) : inv;
}

// PBC: nearest image as in the fp32 kernel, d <- d - L rint(d / L) with rint taken as
// fma(d, 1/L, M) - M, M = 1.5 * 2^52 (PAPER.md:115 footnote 1; reading B2).
template <bool PBC>
__device__ __forceinline__ double min_image_f64(const double d, const PairCoef64& k) {
    if (!PBC) return d;
    return fma(__dsub_rn(fma(d, k.invL, k.magic), k.magic), k.mL, d);
}

// CLAMP: the careful pass of the fp32 kernel (sd_pairs_f32.cuh) in fp64: r^2 is clamped from
// below to k.clampv before 1/r is formed; the true r^2 is returned in r2out.
template <int TENSOR, bool PBC, bool CLAMP>
__device__ __forceinline__ void pair_fast_f64(const double xi, const double yi, const double zi,
                                              const double4 pj, const double4 fj,
                                              const PairCoef64& k, double& px, double& py,
                                              double& pz, float& mn, double& r2out) {
    const double dx = min_image_f64<PBC>(xi - pj.x, k), dy = min_image_f64<PBC>(yi - pj.y, k),
                 dz = min_image_f64<PBC>(zi - pj.z, k);
    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if (CLAMP) {
        r2out = r2;
        r2 = fmax(r2, k.clampv);
    }
    const float r2f = static_cast<float>(r2);
    if (!CLAMP) mn = fminf(mn, r2f);
    const double inv = rsqrt_nr2(r2, r2f);
    const double dF = fma(dz, fj.z, fma(dy, fj.y, dx * fj.x));
    const double inv2 = inv * inv;
    const double inv3 = inv2 * inv;
    double A, Bd;
    if (TENSOR == TENSOR_RPY) {   // folded units (PairCoefT): fj = c1 F_j
        A = fma(k.k2, inv3, inv);
        Bd = fma(k.m3k2, inv2, 1.0) * (inv3 * dF);
    } else {
        A = inv;
        Bd = inv3 * dF;
    }
    px = fma(A, fj.x, px);
    py = fma(A, fj.y, py);
    pz = fma(A, fj.z, pz);
    px = fma(Bd, dx, px);
    py = fma(Bd, dy, py);
    pz = fma(Bd, dz, pz);
}

template <int TENSOR, bool PBC>
__device__ __forceinline__ void pair_exact_f64(const double xi, const double yi, const double zi,
                                               const bool self, const double4 pj,
                                               const double4 fj, const PairCoef64& k, double& px,
                                               double& py, double& pz) {
    if (self) return;
    const double dx = min_image_f64<PBC>(xi - pj.x, k), dy = min_image_f64<PBC>(yi - pj.y, k),
                 dz = min_image_f64<PBC>(zi - pj.z, k);
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if (r2 == 0.0) {
        if (TENSOR == TENSOR_RPY) {
            px = fma(k.mu0r, fj.x, px);
            py = fma(k.mu0r, fj.y, py);
            pz = fma(k.mu0r, fj.z, pz);
        }
        return;
    }
    const double r = sqrt(r2);
    const double inv = 1.0 / r;
    const double dF = fma(dz, fj.z, fma(dy, fj.y, dx * fj.x));
    double A, B;
    if (TENSOR == TENSOR_RPY) {
        if (r2 < k.thr) {
            A = fma(k.ovA, r, k.mu0r);
            B = k.ovB * inv;
        } else {
            const double inv2 = inv * inv;
            const double inv3 = inv2 * inv;
            A = fma(k.k2, inv3, inv);
            B = fma(k.m3k2, inv2, 1.0) * inv3;
        }
    } else {
        A = inv;
        B = inv * inv * inv;
    }
    const double Bd = B * dF;
    px = fma(A, fj.x, px);
    py = fma(A, fj.y, py);
    pz = fma(A, fj.z, pz);
    px = fma(Bd, dx, px);
    py = fma(Bd, dy, py);
    pz = fma(Bd, dz, pz);
}

// the term the CLAMP body added for a pair below the clamp, subtracted again (see the fp32 kernel)
template <int TENSOR, bool PBC>
__device__ __forceinline__ void pair_clamped_sub_f64(const double xi, const double yi,
                                                     const double zi, const double4 pj,
                                                     const double4 fj, const PairCoef64& k,
                                                     double& px, double& py, double& pz) {
    const double dx = min_image_f64<PBC>(xi - pj.x, k), dy = min_image_f64<PBC>(yi - pj.y, k),
                 dz = min_image_f64<PBC>(zi - pj.z, k);
    const double inv = rsqrt_nr2(k.clampv, static_cast<float>(k.clampv));
    const double dF = fma(dz, fj.z, fma(dy, fj.y, dx * fj.x));
    const double inv2 = inv * inv;
    const double inv3 = inv2 * inv;
    double A, Bd;
    if (TENSOR == TENSOR_RPY) {
        A = fma(k.k2, inv3, inv);
        Bd = fma(k.m3k2, inv2, 1.0) * (inv3 * dF);
    } else {
        A = inv;
        Bd = inv3 * dF;
    }
    px = fma(-A, fj.x, px);
    py = fma(-A, fj.y, py);
    pz = fma(-A, fj.z, pz);
    px = fma(-Bd, dx, px);
    py = fma(-Bd, dy, py);
    pz = fma(-Bd, dz, pz);
}

// fp64 counterpart of chunk_fix (sd_pairs_f32.cuh): per particle of the lane, min r^2 over the
// chunk (self pair and pad records excluded); the chunk sums of the particles that have a pair
// below `thr` are recomputed with the exact branching body.  A self pair keeps the clamped term
// A_c F'_i (removed by finalize_f64_kernel).
//   cp / cf : positions / forces of the chunk's records, JS double4 apart from one j to the next
//   ISTEP   : index distance between consecutive particles of a lane
// The work per particle is a real call (__noinline__, operands by value) so that it takes no part
// in the register allocation of the hot loop (sd_pairs_f32.cuh, chunk_fix_group).
struct D3 {
    double x, y, z;
};
template <int TENSOR, bool PBC, int JS>
__device__ __noinline__ D3 chunk_fix_one_f64(const double x, const double y, const double z, const double4* cp,
                                             const double4* cf, const int nj, const int jself, const PairCoef64 k,
                                             const double thr, const D3 base, const D3 cur) {
    double mnq = 1.0e300;
#pragma unroll 4
    for (int jj = 0; jj < nj; ++jj) {
        const double4 pj = cp[jj * JS];
        const double dx = min_image_f64<PBC>(x - pj.x, k), dy = min_image_f64<PBC>(y - pj.y, k),
                     dz = min_image_f64<PBC>(z - pj.z, k);
        const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        mnq = fmin(mnq, jj == jself ? 1.0e300 : r2);
    }
    if (!(mnq < thr)) return cur;
    double nx = 0.0, ny = 0.0, nz = 0.0;
#pragma unroll 1
    for (int jj = 0; jj < nj; ++jj) {
        const double4 pj = cp[jj * JS];
        const double4 fj = cf[jj * JS];
        if (jj == jself) {
            const double ac = self_clamped_coef_f64(TENSOR, k.clampv, k.k2);
            nx = fma(ac, fj.x, nx);
            ny = fma(ac, fj.y, ny);
            nz = fma(ac, fj.z, nz);
        } else {
            pair_exact_f64<TENSOR, PBC>(x, y, z, false, pj, fj, k, nx, ny, nz);
        }
    }
    D3 r;
    r.x = base.x + nx, r.y = base.y + ny, r.z = base.z + nz;
    return r;
}

template <int I, int TENSOR, bool PBC, int JS, int ISTEP>
__device__ __forceinline__ void chunk_fix_f64(const double (&xi)[I], const double (&yi)[I], const double (&zi)[I],
                                              const double4* cp, const double4* cf, const int j0, const int len,
                                              const int N, const int i_first, const PairCoef64& k, const double thr,
                                              double (&px)[I], double (&py)[I], double (&pz)[I],
                                              const double (&qx)[I], const double (&qy)[I], const double (&qz)[I]) {
    const int nj = min(len, N - j0);
#pragma unroll
    for (int m = 0; m < I; ++m) {
        D3 base, cur;
        base.x = qx[m], base.y = qy[m], base.z = qz[m];
        cur.x = px[m], cur.y = py[m], cur.z = pz[m];
        const D3 r = chunk_fix_one_f64<TENSOR, PBC, JS>(xi[m], yi[m], zi[m], cp, cf, nj, i_first + m * ISTEP - j0, k,
                                                        thr, base, cur);
        px[m] = r.x, py[m] = r.y, pz[m] = r.z;
    }
}

template <int I, int TENSOR, bool PBC, int TJ = kTJ64>
__global__ void __launch_bounds__(kThreads, (I == 1) ? 3 : ((I == 2) ? 2 : 1))
pairs_f64_kernel(const double4* __restrict__ rec, double4* __restrict__ part, const Schedule sch,
                 const PairCoef64 k, const float thr, const int N, const long long slot_stride) {
    constexpr int IB = kThreads * I;
    __shared__ __align__(128) double4 tiles[kStages][TJ * 2];
    __shared__ __align__(8) uint64_t full_bar[kStages];
    __shared__ __align__(8) uint64_t empty_bar[kStages];

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int c = sch.cta_piece[blockIdx.x];  // pieces of one SM's CTAs are consecutive (balance)
    const long long u_begin = sch.cta_u0[c];
    const long long u_end = sch.cta_u0[c + 1];
    const int n_units = static_cast<int>(u_end - u_begin);
    const int T = sch.T;

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], kWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    int pf_n = 0;
    int pf_t = static_cast<int>(u_begin % T);
    auto produce = [&]() {
        const int s = pf_n % kStages;
        const int q = pf_n / kStages;
        if (q > 0) mbar_wait(&empty_bar[s], (q - 1) & 1);
        mbar_arrive_expect_tx(&full_bar[s], TJ * 64);
        bulk_load(&tiles[s][0], rec + static_cast<size_t>(pf_t) * (TJ * 2), TJ * 64,
                  &full_bar[s]);
        ++pf_n;
        if (++pf_t == T) pf_t = 0;
    };
    if (tid == 0) {
        for (int q = 0; q < kPrefetch && pf_n < n_units; ++q) produce();
    }

    int n = 0;
    long long u = u_begin;
    while (u < u_end) {
        const int b = static_cast<int>(u / T);
        const int t0 = static_cast<int>(u - static_cast<long long>(b) * T);
        const long long left = u_end - u;
        const int nt = (left < static_cast<long long>(T - t0)) ? static_cast<int>(left) : (T - t0);
        const int i_first = b * IB + tid;

        double xi[I], yi[I], zi[I], px[I], py[I], pz[I];
#pragma unroll
        for (int m = 0; m < I; ++m) {
            const int i = i_first + m * kThreads;
            const double dm = static_cast<double>(SD_DUMMY_I_POS);
            const double4 p = (i < N) ? rec[2 * static_cast<size_t>(i)] : make_double4(dm, dm, dm, 0.0);
            xi[m] = p.x;
            yi[m] = p.y;
            zi[m] = p.z;
            px[m] = py[m] = pz[m] = 0.0;
        }

        for (int tt = 0; tt < nt; ++tt, ++n) {
            if (tid == 0 && pf_n < n_units) produce();
            const int s = n % kStages;
            mbar_wait(&full_bar[s], (n / kStages) & 1);
            const double4* tile = &tiles[s][0];
            const int jbase = (t0 + tt) * TJ;

#pragma unroll 1
            for (int ch = 0; ch < TJ / kChunk; ++ch) {
                const double4* cj = tile + ch * (kChunk * 2);
                double qx[I], qy[I], qz[I];
#pragma unroll
                for (int m = 0; m < I; ++m) {
                    qx[m] = px[m];
                    qy[m] = py[m];
                    qz[m] = pz[m];
                }
                float mn = 3.0e38f;
                double r2t;
                const int j0 = jbase + ch * kChunk;
                const int rel = j0 - (i_first - lane);  // chunk holding this warp's own particles?
                const bool diag = rel >= 0 && (rel % kThreads) == 0 && rel < I * kThreads;
                bool fix;
                if (!diag) {
#pragma unroll 4
                    for (int jj = 0; jj < kChunk; ++jj) {
                        const double4 pj = cj[2 * jj];
                        const double4 fj = cj[2 * jj + 1];
#pragma unroll
                        for (int m = 0; m < I; ++m)
                            pair_fast_f64<TENSOR, PBC, false>(xi[m], yi[m], zi[m], pj, fj, k, px[m],
                                                              py[m], pz[m], mn, r2t);
                    }
                    fix = mn < thr;
                } else {
                    // diagonal chunk: clamped body, branch-free; exact unless a pair other than the
                    // lane's self pair lies below the clamp (see the fp32 kernel)
                    int zeros = 0;
#pragma unroll 4
                    for (int jj = 0; jj < kChunk; ++jj) {
                        const double4 pj = cj[2 * jj];
                        const double4 fj = cj[2 * jj + 1];
#pragma unroll
                        for (int m = 0; m < I; ++m) {
                            pair_fast_f64<TENSOR, PBC, true>(xi[m], yi[m], zi[m], pj, fj, k, px[m],
                                                             py[m], pz[m], mn, r2t);
                            const bool z = r2t == 0.0;
                            zeros += z ? 1 : 0;
                            mn = fminf(mn, z ? 3.0e38f : static_cast<float>(r2t));
                        }
                    }
                    fix = mn < static_cast<float>(k.clampv) * 1.000001f || zeros != ((j0 + lane < N) ? 1 : 0);
                }
                if (fix)  // rare: repair the sums of the particles that have a pair below the clamp
                    chunk_fix_f64<I, TENSOR, PBC, 2, kThreads>(xi, yi, zi, cj, cj + 1, j0, kChunk, N, i_first, k,
                                                               diag ? k.clampv : k.thr, px, py, pz, qx, qy, qz);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[s]);
        }

        const int slot = c - sch.blk_first_cta[b];
        double4* out = part + static_cast<size_t>(slot) * slot_stride;
#pragma unroll
        for (int m = 0; m < I; ++m) {
            const int i = i_first + m * kThreads;
            if (i < N) out[i] = make_double4(px[m], py[m], pz[m], 0.0);
        }
        u += nt;
    }
}

}  // namespace sd
