// sd_pairs_f64w.cuh -- the warp-split one-launch kernel (sd_pairs_f32w.cuh) in fp64.
//
// Same mapping: all 8 warps of a CTA own the same 32 I particles (I = 4 per lane, 128-particle
// i-blocks, one CTA per SM), the flattened (i-block, j) space is cut at 4-j granularity into one
// equal piece per CTA, every warp takes an eighth of its CTA's piece through its own bulk-copy pipeline,
// the warps' sums are combined through shared memory in warp order, and the CTA that delivers the
// last partial of an i-block finishes its rows (self term, clamped self-pair term out, velocity,
// fused integrator update).  Reads the caller's pos / force arrays; no pack, no finalize launch.
// Arithmetic: the scalar fp64 bodies of sd_pairs_f64.cuh (25 fp64 instructions per pair), plain
// fp64 sums, branch-free diagonal chunks, chunk_fix_f64 for chunks with a pair below the clamp.
#pragma once
#include "sd_common.cuh"
#include "sd_pairs_f32w.cuh"
#include "sd_pairs_f64.cuh"
#include "sd_stream.cuh"

namespace sd {

constexpr int kW64SJ = 32;     // j records (2 x 32 bytes each) per warp-private sub-tile
// Measured (profiles/r02_mid_n.md): against the one-launch warp-per-particle kernel it wins from N = 1024 on
// (14.6 / 20.9 / 28.1 / 35.0 us at N = 1024 / 1536 / 2048 / 2560 against 16.6 / 24.9 / 33.0 / 59.6), against the classic
// fp64 kernels (1 - 2 particles per thread, 2 - 3 CTAs per SM) per product up to N = 3000 (43.3 against 47.3 us) but not per
// Euler step there (41.9 against 39.6 us: sd_step never runs the pack kernel); from N = 4096 on it
// loses (69.9 / 167.5 / 537 us at 4096 / 8192 / 16384 against 61.7 / 162 / 517: two warps per scheduler do not hide the
// DFMA latency that 24 resident warps hide).  Default range: kW64MinN < N <= kW64MaxN.
constexpr int kW64MinN = 1000;
constexpr int kW64MaxN = 2800;

struct FinArgs64 {
    double4* vel;
    const double4* pos_base;
    double4* pos_out;
    double dt;
    double c1;
    double mu0;
    int mode;
};

template <int I>
struct W64Shape {
    static constexpr int IBW = 32 * I;
    static constexpr size_t tile_bytes = static_cast<size_t>(kWarps) * kWStages * kW64SJ * 2 * sizeof(double4);
    static constexpr size_t red_bytes = static_cast<size_t>(kWarps) * 3 * IBW * sizeof(double);
    static constexpr size_t smem_bytes = tile_bytes + red_bytes;
};

template <int I, int TENSOR, bool PBC>
__global__ void __launch_bounds__(kThreads, 1)
pairs_f64w_kernel(const double4* __restrict__ pos, const double4* __restrict__ frc,
                  const double4* __restrict__ padblk, double4* __restrict__ part,
                  int* __restrict__ blk_done, const Schedule sch, const PairCoef64 k, const float thr,
                  const FinArgs64 fin, const int N, const long long slot_stride) {
    typedef W64Shape<I> W;
    constexpr int IBW = W::IBW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* red = reinterpret_cast<double*>(smem_raw + W::tile_bytes);  // [kWarps][3][IBW]
    __shared__ __align__(8) uint64_t full_bar[kWarps][kWStages];
    __shared__ int s_last;

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    double4* wtiles = reinterpret_cast<double4*>(smem_raw) + static_cast<size_t>(warp) * (kWStages * 2 * kW64SJ);
    const int c = blockIdx.x;  // piece = blockIdx.x; cut points g U / G as in build_schedule (sd_b200.cu)
    const int T = sch.T;
    const long long U = static_cast<long long>(sch.B) * T;
    const long long u_begin = static_cast<long long>(c) * U / sch.G;
    const long long u_end = static_cast<long long>(c + 1) * U / sch.G;

    if (lane == 0) {
        for (int s = 0; s < kWStages; ++s) mbar_init(&full_bar[warp][s], 1);
        mbar_fence_init();
    }
    __syncwarp();

    int wn = 0;
    long long u = u_begin;
    while (u < u_end) {
        const int b = static_cast<int>(u / T);
        const int t0 = static_cast<int>(u - static_cast<long long>(b) * T);
        const long long left = u_end - u;
        const int nt = (left < static_cast<long long>(T - t0)) ? static_cast<int>(left) : (T - t0);
        const int i_blk = b * IBW;
        const int i_first = i_blk + lane;  // the lane's particles: i_first + 32 m
        const int per = (nt + kWarps - 1) / kWarps;
        const int q_lo = min(t0 + warp * per, t0 + nt), q_hi = min(q_lo + per, t0 + nt);
        const int j_lo = q_lo * kWQ, j_hi = q_hi * kWQ;
        const int nsub = (j_hi - j_lo + kW64SJ - 1) / kW64SJ;

        auto produce = [&](const int ks) {
            const int s = (wn + ks) % kWStages;
            double4* dst = wtiles + s * (2 * kW64SJ);
            const int j0 = j_lo + ks * kW64SJ;
            const int cnt = min(kW64SJ, j_hi - j0);
            const int valid = max(0, min(cnt, N - j0));
            fence_proxy_async();
            mbar_arrive_expect_tx(&full_bar[warp][s], cnt * 64);
            if (valid > 0) {
                bulk_load(dst, pos + j0, valid * 32, &full_bar[warp][s]);
                bulk_load(dst + kW64SJ, frc + j0, valid * 32, &full_bar[warp][s]);
            }
            if (valid < cnt) {
                bulk_load(dst + valid, padblk, (cnt - valid) * 32, &full_bar[warp][s]);
                bulk_load(dst + kW64SJ + valid, padblk + kW64SJ, (cnt - valid) * 32, &full_bar[warp][s]);
            }
        };
        if (lane == 0) {
            for (int ks = 0; ks < kWStages - 1 && ks < nsub; ++ks) produce(ks);
        }

        double xi[I], yi[I], zi[I], px[I], py[I], pz[I];
#pragma unroll
        for (int m = 0; m < I; ++m) {
            const int i = i_first + 32 * m;
            const double dm = static_cast<double>(SD_DUMMY_I_POS);
            const double4 p = (i < N) ? pos[i] : make_double4(dm, dm, dm, 0.0);
            xi[m] = p.x, yi[m] = p.y, zi[m] = p.z;
            px[m] = py[m] = pz[m] = 0.0;
        }

#pragma unroll 1
        for (int ks = 0; ks < nsub; ++ks) {
            const int s = (wn + ks) % kWStages;
            __syncwarp();
            if (lane == 0 && ks + kWStages - 1 < nsub) produce(ks + kWStages - 1);
            mbar_wait(&full_bar[warp][s], ((wn + ks) / kWStages) & 1);
            const double4* cp = wtiles + s * (2 * kW64SJ);  // positions; forces kW64SJ further
            const double4* cf = cp + kW64SJ;
            const int j0 = j_lo + ks * kW64SJ;
            const int len = min(kW64SJ, j_hi - j0);         // one compensation-free chunk, multiple of 4
            double qx[I], qy[I], qz[I];
#pragma unroll
            for (int m = 0; m < I; ++m) qx[m] = px[m], qy[m] = py[m], qz[m] = pz[m];
            float mn = 3.0e38f;
            double r2t;
            const bool diag = (j0 + len > i_blk) && (j0 < i_blk + IBW);
            bool fix;
            if (!diag) {
#pragma unroll 1
                for (int jq = 0; jq < len; jq += kWQ) {
#pragma unroll
                    for (int jj = 0; jj < kWQ; ++jj) {
                        const double4 pj = cp[jq + jj];
                        const double4 fj = cf[jq + jj];
#pragma unroll
                        for (int m = 0; m < I; ++m)
                            pair_fast_f64<TENSOR, PBC, false>(xi[m], yi[m], zi[m], pj, fj, k, px[m], py[m], pz[m],
                                                              mn, r2t);
                    }
                }
                fix = mn < thr;
            } else {
                int zeros = 0;
#pragma unroll 1
                for (int jq = 0; jq < len; jq += kWQ) {
#pragma unroll
                    for (int jj = 0; jj < kWQ; ++jj) {
                        const double4 pj = cp[jq + jj];
                        const double4 fj = cf[jq + jj];
#pragma unroll
                        for (int m = 0; m < I; ++m) {
                            pair_fast_f64<TENSOR, PBC, true>(xi[m], yi[m], zi[m], pj, fj, k, px[m], py[m], pz[m],
                                                             mn, r2t);
                            const bool z = r2t == 0.0;
                            zeros += z ? 1 : 0;
                            mn = fminf(mn, z ? 3.0e38f : static_cast<float>(r2t));
                        }
                    }
                }
                const int first = j0 > i_first ? i_first + ((j0 - i_first + 31) & ~31) : i_first;
                const bool mine = first < j0 + len && first < i_blk + IBW && first < N;
                fix = mn < static_cast<float>(k.clampv) * 1.000001f || zeros != (mine ? 1 : 0);
            }
            if (fix)
                chunk_fix_f64<I, TENSOR, PBC, 1, 32>(xi, yi, zi, cp, cf, j0, len, N, i_first, k,
                                                     diag ? k.clampv : k.thr, px, py, pz, qx, qy, qz);
        }
        wn += nsub;

        // ---- combine the warps' sums in warp order: one partial per particle and segment --------
#pragma unroll
        for (int m = 0; m < I; ++m) {
            double* r0 = red + (warp * 3) * IBW + 32 * m + lane;
            r0[0 * IBW] = px[m], r0[1 * IBW] = py[m], r0[2 * IBW] = pz[m];
        }
        __syncthreads();
        const int slot = c - sch.blk_first_cta[b];
        const int nslots = sch.blk_nslots[b];
        const int i_mine = i_blk + tid;  // the particle this thread reduces (tid < IBW)
        double vx = 0.0, vy = 0.0, vz = 0.0;
        if (tid < IBW) {
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const double* r0 = red + (w * 3) * IBW + tid;
                vx += r0[0 * IBW], vy += r0[1 * IBW], vz += r0[2 * IBW];
            }
        }
        bool last = true;
        if (nslots > 1) {
            if (tid < IBW && i_mine < N)
                part[static_cast<size_t>(slot) * slot_stride + i_mine] = make_double4(vx, vy, vz, 0.0);
            __threadfence();
            __syncthreads();
            if (tid == 0) s_last = (atomicAdd(&blk_done[b], 1) == nslots - 1);
            __syncthreads();
            last = s_last != 0;
        }
        if (last) {  // the CTA that delivered the last partial of this i-block finishes its rows
            if (nslots > 1) {
                __threadfence();
                if (tid == 0) blk_done[b] = 0;
                vx = vy = vz = 0.0;
                if (tid < IBW && i_mine < N) {
                    for (int s0 = 0; s0 < nslots; s0 += kFinBatch) {
                        double2 a[kFinBatch];
                        double bz[kFinBatch];
#pragma unroll
                        for (int q = 0; q < kFinBatch; ++q) {
                            if (s0 + q < nslots) {
                                const double* p = reinterpret_cast<const double*>(
                                    part + static_cast<size_t>(s0 + q) * slot_stride + i_mine);
                                a[q] = __ldcg(reinterpret_cast<const double2*>(p));
                                bz[q] = __ldcg(p + 2);
                            }
                        }
#pragma unroll
                        for (int q = 0; q < kFinBatch; ++q) {
                            if (s0 + q < nslots) vx += a[q].x, vy += a[q].y, vz += bz[q];
                        }
                    }
                }
            }
            if (tid < IBW && i_mine < N) {
                const double4 f = frc[i_mine];
                const double ac = self_clamped_coef_f64(TENSOR, k.clampv, k.k2);
                vx = fin.mu0 * f.x + fin.c1 * (vx - ac * f.x);
                vy = fin.mu0 * f.y + fin.c1 * (vy - ac * f.y);
                vz = fin.mu0 * f.z + fin.c1 * (vz - ac * f.z);
                fin.vel[i_mine] = make_double4(vx, vy, vz, 0.0);
                if (fin.mode != FIN_VEL) {
                    const double4 p0 = fin.pos_base[i_mine];
                    const double h = (fin.mode == FIN_HALF) ? 0.5 * fin.dt : fin.dt;
                    fin.pos_out[i_mine] = make_double4(p0.x + h * vx, p0.y + h * vy, p0.z + h * vz, 0.0);
                }
            }
        }
        __syncthreads();  // `red` and `s_last` are reused by the next segment
        u += nt;
    }
}

}  // namespace sd
