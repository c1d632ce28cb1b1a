// sd_pairs_f32w.cuh -- all-pairs mobility kernel, fp32, j split across the WARPS of a CTA, whole
// product in ONE launch (no pack kernel, no finalize kernel).
//
// Same pair arithmetic as sd_pairs_f32.cuh (packed FFMA2 body, chunked Kahan, clamped careful
// pass); what differs is the mapping, made for the under-filled regime N ~ 3e3 ... 1e5
// (PAPER.md:239, :273), where the classic kernel needs 2048-particle i-blocks to run its best
// inner loop and then has too few, too coarse work units for 148 SMs:
//  * all 8 warps of a CTA own the SAME 32 * 2 I2 particles i (8 per lane with I2 = 4, the inner
//    loop of the large-N kernel) and split the CTA's j range between them: the flattened
//    (i-block, j) space is cut at a granularity of 4 j into one equal piece per SM ("stream-K"),
//    and every warp takes an eighth of its CTA's piece -- the split is exact to 4 j per warp at
//    any N.  An i-block is 256 particles instead of 2048, so the per-block tail (diagonal chunks,
//    repairs) shrinks by the same factor;
//  * every warp runs its own pipeline of bulk copies (cp.async.bulk + one mbarrier per stage,
//    three 64-record sub-tiles in flight / in use per warp): no barrier is shared between warps
//    inside a segment, a warp that repairs a chunk delays nobody;
//  * the Kahan pairs (s, c) live in shared memory (touched once per 32 j), 48 registers less;
//  * diagonal chunks run the clamped body branch-free and count exact zeros; a chunk that met a
//    pair below the clamp repairs only the packed groups concerned (chunk_fix);
//  * the warps' compensated sums are combined through shared memory in fp64 in warp order, and
//    the CTA writes ONE (hi, lo) partial per particle and segment;
//  * the kernel reads the caller's pos / force arrays directly (two bulk copies per sub-tile, laid
//    out {64 positions | 64 forces}; the ragged tail of the system comes from a context-owned
//    block of pad records), works in the folded units of sd_common.cuh on the RAW
//    forces and multiplies by c1 = mu0 3a/4 at the very end;
//  * the last CTA to deliver a partial of an i-block (a ticket counter per block; the sum itself
//    runs over the slots in fixed order, so the result does not depend on who is last) adds the
//    slots in fp64, the self term mu0 F_i, takes the clamped self-pair term out again
//    (self_clamped_coef), writes vel and applies the fused integrator update -- the whole of
//    SURVEY 8(a) a1-a5 in one launch.
#pragma once
#include "sd_common.cuh"
#include "sd_pairs_f32.cuh"
#include "sd_stream.cuh"

namespace sd {

// Up to here the warp-split kernel runs by default (measured against the classic kernels with
// `python bench.py --n N --jsplit classic|warp --launches-per-step K`, CUDA-graph replay,
// profiles/r02_mid_n.md: free space 11 % faster at N = 4096, 5 % at 8192, 6 % at 16 384 and 20 480,
// 2 % at 24 576, 2 % slower at 32 768; periodic box 10 % at 4096, 2 % at 8192, within 1.6 % of each
// other from 12 288 to 24 576).
constexpr int kWMaxN = 28000;
constexpr int kWMaxNBox = 14000;

// everything the fused epilogue needs
struct FinArgs {
    float4* vel;             // out: velocities of this product
    const float4* pos_base;  // r_n (high words) the update starts from      (mode != FIN_VEL)
    float4* pos_lo;          // low words of r_n, rewritten by FIN_EULER / FIN_FULL
    float4* pos_out;         // where the new positions go (never the array the pairs are read from)
    double dt;
    double c1;               // mu0 3a/4: the partial sums are in units of 1 / c1
    double mu0;
    int mode;                // FIN_VEL / FIN_EULER / FIN_HALF / FIN_FULL
    int pos_comp;
};

constexpr int kWQ = 4;        // schedule granule: j records per "quad" (= the unrolled loop body)
constexpr int kWSJ = 64;      // j records per warp-private sub-tile (two compensation chunks; 128: +0.5 % at N >= 16384, -1 % at 4096)
constexpr int kWStages = 3;   // sub-tiles per warp in flight / in use

template <int I2>
struct WShape {
    static constexpr int IBW = 64 * I2;  // particles per i-block: 32 lanes x 2 I2
    static constexpr size_t tile_bytes = static_cast<size_t>(kWarps) * kWStages * kWSJ * 2 * sizeof(float4);
    static constexpr size_t red_bytes = static_cast<size_t>(kWarps) * 6 * IBW * sizeof(float);
    static constexpr size_t smem_bytes = tile_bytes + red_bytes;
};

#ifdef SD_W_TRACE  // per-CTA timeline for tuning; not part of the product build
__device__ unsigned long long g_wtrace[1024 * 8];
__device__ __forceinline__ void wtrace(const int slot) {
    if (threadIdx.x == 0 && blockIdx.x < 1024) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
        g_wtrace[blockIdx.x * 8 + slot] = t;
    }
}
#define SD_WTRACE(slot) wtrace(slot)
#else
#define SD_WTRACE(slot)
#endif

__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

template <int I2, int TENSOR, int ACC, bool PBC>
__global__ void __launch_bounds__(kThreads, (I2 == 4) ? 1 : 2)
pairs_f32w_kernel(const float4* __restrict__ pos, const float4* __restrict__ frc,
                  const float4* __restrict__ padblk, float4* __restrict__ part,
                  int* __restrict__ blk_done, const Schedule sch, const PairCoef k, const FinArgs fin,
                  const int N, const long long slot_stride) {
    typedef WShape<I2> W;
    constexpr int IBW = W::IBW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* red = reinterpret_cast<float*>(smem_raw + W::tile_bytes);      // [kWarps][6][IBW]
    __shared__ __align__(8) uint64_t full_bar[kWarps][kWStages];
    __shared__ int s_last;

    SD_WTRACE(0);
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    // this warp's private ring of sub-tiles, each laid out {kWSJ positions | kWSJ forces}
    float4* wtiles = reinterpret_cast<float4*>(smem_raw) + static_cast<size_t>(warp) * (kWStages * 2 * kWSJ);
    // one CTA per SM, piece = blockIdx.x; the cut points g U / G of build_schedule (sd_b200.cu) are
    // recomputed here instead of loaded: two dependent global loads less before the first copy
    const int c = blockIdx.x;
    const int T = sch.T;  // quads per row of the (i-block, quad) grid
    const long long U = static_cast<long long>(sch.B) * T;
    const long long u_begin = static_cast<long long>(c) * U / sch.G;
    const long long u_end = static_cast<long long>(c + 1) * U / sch.G;

    if (lane == 0) {
        for (int s = 0; s < kWStages; ++s) mbar_init(&full_bar[warp][s], 1);
        mbar_fence_init();
    }
    __syncwarp();

    int wn = 0;  // sub-tiles this warp has consumed so far (ring position and barrier phase)
    long long u = u_begin;
    while (u < u_end) {
        const int b = static_cast<int>(u / T);
        const int t0 = static_cast<int>(u - static_cast<long long>(b) * T);
        const long long left = u_end - u;
        const int nt = (left < static_cast<long long>(T - t0)) ? static_cast<int>(left) : (T - t0);
        const int i_blk = b * IBW;
        const int i_first = i_blk + lane;  // particle of (m = 0, half 0); the others follow in steps of 32
        // this warp's share of the segment: a contiguous run of quads, the same number (+-1) for
        // every warp: the split of the work is exact to 4 j per warp whatever N
        const int per = (nt + kWarps - 1) / kWarps;
        const int q_lo = min(t0 + warp * per, t0 + nt), q_hi = min(q_lo + per, t0 + nt);
        const int j_lo = q_lo * kWQ, j_hi = q_hi * kWQ;      // records [j_lo, j_hi); those >= N are pads
        const int nsub = (j_hi - j_lo + kWSJ - 1) / kWSJ;

        auto produce = [&](const int ks) {  // lane 0: fetch sub-tile ks of this warp's run
            const int s = (wn + ks) % kWStages;
            float4* dst = wtiles + s * (2 * kWSJ);
            const int j0 = j_lo + ks * kWSJ;
            const int cnt = min(kWSJ, j_hi - j0);
            const int valid = max(0, min(cnt, N - j0));
            fence_proxy_async();  // the generic-proxy reads of the stage's previous tenant are done
            mbar_arrive_expect_tx(&full_bar[warp][s], cnt * 32);
            if (valid > 0) {
                bulk_load(dst, pos + j0, valid * 16, &full_bar[warp][s]);
                bulk_load(dst + kWSJ, frc + j0, valid * 16, &full_bar[warp][s]);
            }
            if (valid < cnt) {  // ragged tail of the system: pad records (far away, zero force)
                bulk_load(dst + valid, padblk, (cnt - valid) * 16, &full_bar[warp][s]);
                bulk_load(dst + kWSJ + valid, padblk + kWSJ, (cnt - valid) * 16, &full_bar[warp][s]);
            }
        };
        if (lane == 0) {
            for (int ks = 0; ks < kWStages - 1 && ks < nsub; ++ks) produce(ks);
        }

        f32x2 xi[I2], yi[I2], zi[I2];
#pragma unroll
        for (int m = 0; m < I2; ++m) {
            const int i0 = i_first + 64 * m;
            const int i1 = i0 + 32;
            const float4 d = make_float4(SD_DUMMY_I_POS, SD_DUMMY_I_POS, SD_DUMMY_I_POS, 0.f);
            const float4 p0 = (i0 < N) ? pos[i0] : d;
            const float4 p1 = (i1 < N) ? pos[i1] : d;
            const f32x2 zero = bc2(0.f);
            xi[m] = add2(pk2(p0.x, p1.x), zero);
            yi[m] = add2(pk2(p0.y, p1.y), zero);
            zi[m] = add2(pk2(p0.z, p1.z), zero);
        }
        // The Kahan pairs (s, c) of the lane's particles live in shared memory, in the very array
        // the cross-warp combine reads afterwards: they are touched once per chunk of 32 j, and 48
        // registers less in the hot loop is what keeps it free of spills and copies.  Element
        // (warp, component, m, lane) is one f32x2 = the two particles of packed group m.
        f32x2* kst = reinterpret_cast<f32x2*>(red) + (warp * 6) * (IBW / 2) + lane;
        f32x2 px[I2], py[I2], pz[I2];
#pragma unroll
        for (int m = 0; m < I2; ++m) {
#pragma unroll
            for (int comp = 0; comp < 6; ++comp) kst[comp * (IBW / 2) + 32 * m] = bc2(0.f);
            px[m] = py[m] = pz[m] = bc2(0.f);
        }

#pragma unroll 1
        for (int ks = 0; ks < nsub; ++ks) {
            const int s = (wn + ks) % kWStages;
            __syncwarp();
            if (lane == 0 && ks + kWStages - 1 < nsub) produce(ks + kWStages - 1);
            mbar_wait(&full_bar[warp][s], ((wn + ks) / kWStages) & 1);
            if (ks == 0 && u == u_begin) SD_WTRACE(1);
            const float4* tp = wtiles + s * (2 * kWSJ);
            const int jt = j_lo + ks * kWSJ;
            const int cnt = min(kWSJ, j_hi - jt);
#pragma unroll 1
            for (int c0 = 0; c0 < cnt; c0 += kChunk) {
            const int len = min(kChunk, cnt - c0);      // records of this compensation chunk (multiple of 4)
            const float4* cp = tp + c0;                 // positions
            const float4* cf = cp + kWSJ;               // forces
            const int j0 = jt + c0;
            f32x2 qx[I2], qy[I2], qz[I2];
#pragma unroll
            for (int m = 0; m < I2; ++m) {
                if (ACC == ACC_KAHAN) {
                    px[m] = py[m] = pz[m] = bc2(0.f);
                } else {
                    qx[m] = px[m];
                    qy[m] = py[m];
                    qz[m] = pz[m];
                }
            }
            float mn = 3.0e38f;  // unused: min r^2 is tracked per packed group
            float mng[I2];
#pragma unroll
            for (int m = 0; m < I2; ++m) mng[m] = 3.0e38f;
            float r2v[2 * I2];
            // does this chunk hold self pairs (j = i) of the warp's particles?
            const bool diag = (j0 + len > i_blk) && (j0 < i_blk + IBW);
            unsigned groups = 0u;  // packed groups whose chunk sum has to be repaired
            if (!diag) {
                if (len == kChunk) {  // the common case, with a compile-time trip count
#pragma unroll kUnrollJ
                    for (int jj = 0; jj < kChunk; ++jj) {
                        const float4 pj = cp[jj];
                        const float4 fj = cf[jj];
                        pair_fast_staged<I2, TENSOR, PBC, false, true>(xi, yi, zi, pj, fj, k, px, py, pz, mn,
                                                                       r2v, mng);
                    }
                } else {
#pragma unroll 1
                    for (int jq = 0; jq < len; jq += kWQ) {
#pragma unroll
                        for (int jj = 0; jj < kWQ; ++jj) {
                            const float4 pj = cp[jq + jj];
                            const float4 fj = cf[jq + jj];
                            pair_fast_staged<I2, TENSOR, PBC, false, true>(xi, yi, zi, pj, fj, k, px, py, pz,
                                                                           mn, r2v, mng);
                        }
                    }
                }
#pragma unroll
                for (int m = 0; m < I2; ++m) groups |= (mng[m] < k.thr ? 1u : 0u) << m;
            } else {
                // diagonal chunk: the clamped body, branch-free (a self pair adds the finite term
                // A_c F'_i that the epilogue removes).  It is exact unless a pair other than the
                // self pairs lies below the clamp: min r^2 per group over the pairs with r^2 > 0,
                // and the number of exact zeros against the number of self pairs this lane meets.
                int zeros = 0;
#pragma unroll 1
                for (int jq = 0; jq < len; jq += kWQ) {
#pragma unroll
                    for (int jj = 0; jj < kWQ; ++jj) {
                        const float4 pj = cp[jq + jj];
                        const float4 fj = cf[jq + jj];
                        pair_fast_staged<I2, TENSOR, PBC, true>(xi, yi, zi, pj, fj, k, px, py, pz, mn, r2v);
#pragma unroll
                        for (int q = 0; q < 2 * I2; ++q) {
                            const bool z = r2v[q] == 0.f;
                            zeros += z ? 1 : 0;
                            mng[q / 2] = fminf(mng[q / 2], z ? 3.0e38f : r2v[q]);
                        }
                    }
                }
                // the lane's particles are i_first + 32 q: at most one of them lies in [j0, j0 + len)
                const int first = j0 > i_first ? i_first + ((j0 - i_first + 31) & ~31) : i_first;
                const bool mine = first < j0 + len && first < i_blk + IBW && first < N;
#pragma unroll
                for (int m = 0; m < I2; ++m) groups |= (mng[m] < k.clampv ? 1u : 0u) << m;
                if (zeros != (mine ? 1 : 0)) groups = (1u << I2) - 1u;  // coincident centres: all groups
            }
            if (groups) {  // rare: repair the chunk sums of the groups that met a pair below the clamp
#pragma unroll
                for (int m = 0; m < I2; ++m) {
                    if ((groups >> m) & 1u) {
                        P3 base;
                        base.x = ACC == ACC_KAHAN ? bc2(0.f) : qx[m];
                        base.y = ACC == ACC_KAHAN ? bc2(0.f) : qy[m];
                        base.z = ACC == ACC_KAHAN ? bc2(0.f) : qz[m];
                        const P3 r = chunk_fix_group<TENSOR, PBC, 1, 32>(xi[m], yi[m], zi[m], cp, cf, j0, len, N,
                                                                         i_first + 64 * m, k, base);
                        px[m] = r.x, py[m] = r.y, pz[m] = r.z;
                    }
                }
            }
            if (ACC == ACC_KAHAN) {
#pragma unroll
                for (int m = 0; m < I2; ++m) {
                    f32x2* e = kst + 32 * m;
                    f32x2 s0 = e[0 * (IBW / 2)], s1 = e[1 * (IBW / 2)], s2 = e[2 * (IBW / 2)];
                    f32x2 c0k = e[3 * (IBW / 2)], c1k = e[4 * (IBW / 2)], c2k = e[5 * (IBW / 2)];
                    kahan_merge2(s0, c0k, px[m]);
                    kahan_merge2(s1, c1k, py[m]);
                    kahan_merge2(s2, c2k, pz[m]);
                    e[0 * (IBW / 2)] = s0, e[1 * (IBW / 2)] = s1, e[2 * (IBW / 2)] = s2;
                    e[3 * (IBW / 2)] = c0k, e[4 * (IBW / 2)] = c1k, e[5 * (IBW / 2)] = c2k;
                }
            }
            }  // chunks
        }
        wn += nsub;
        if (u == u_begin) SD_WTRACE(2);

        // ---- combine the warps' sums (fp64, warp order): one (hi, lo) partial per particle ----
        if (ACC == ACC_PLAIN) {  // the running sums are the result; compensation words stay 0
#pragma unroll
            for (int m = 0; m < I2; ++m) {
                kst[0 * (IBW / 2) + 32 * m] = px[m];
                kst[1 * (IBW / 2) + 32 * m] = py[m];
                kst[2 * (IBW / 2) + 32 * m] = pz[m];
            }
        }
        __syncthreads();
        const int slot = c - sch.blk_first_cta[b];
        const int nslots = sch.blk_nslots[b];
        // float t of a component row belongs to packed group t / 64, lane (t % 64) / 2, half t % 2
        const int i_mine = i_blk + 64 * (tid >> 6) + 32 * (tid & 1) + ((tid & 63) >> 1);  // tid < IBW
        double vx = 0.0, vy = 0.0, vz = 0.0;
        if (tid < IBW) {
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const float* r0 = red + (w * 6) * IBW + tid;
                vx += static_cast<double>(r0[0 * IBW]) - static_cast<double>(r0[3 * IBW]);
                vy += static_cast<double>(r0[1 * IBW]) - static_cast<double>(r0[4 * IBW]);
                vz += static_cast<double>(r0[2 * IBW]) - static_cast<double>(r0[5 * IBW]);
            }
        }
        if (u == u_begin) SD_WTRACE(3);
        bool last = true;
        if (nslots > 1) {
            if (tid < IBW && i_mine < N) {
                const float hx = static_cast<float>(vx), hy = static_cast<float>(vy), hz = static_cast<float>(vz);
                float4* out = part + (static_cast<size_t>(slot) * slot_stride + i_mine) * 2;
                out[0] = make_float4(hx, hy, hz, 0.f);
                out[1] = make_float4(static_cast<float>(static_cast<double>(hx) - vx),
                                     static_cast<float>(static_cast<double>(hy) - vy),
                                     static_cast<float>(static_cast<double>(hz) - vz), 0.f);
            }
            __threadfence();
            __syncthreads();
            if (tid == 0) s_last = (atomicAdd(&blk_done[b], 1) == nslots - 1);
            __syncthreads();
            last = s_last != 0;
        }
        if (u == u_begin) SD_WTRACE(4);
        // ---- the CTA that delivered the last partial of this i-block finishes its rows ----------
        if (last) {
            if (nslots > 1) {
                __threadfence();
                if (tid == 0) blk_done[b] = 0;  // ready for the next launch
                vx = vy = vz = 0.0;
                if (tid < IBW && i_mine < N) {
                    for (int s0 = 0; s0 < nslots; s0 += kFinBatch) {
                        float4 hi[kFinBatch], lo[kFinBatch];
#pragma unroll
                        for (int q = 0; q < kFinBatch; ++q) {
                            if (s0 + q < nslots) {
                                const float4* p = part + (static_cast<size_t>(s0 + q) * slot_stride + i_mine) * 2;
                                hi[q] = __ldcg(p);
                                lo[q] = __ldcg(p + 1);
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
                }
            }
            if (tid < IBW && i_mine < N) {
                const float4 f = frc[i_mine];
                // v = mu0 F_i + c1 (sum - A_c F_i): self term in, clamped self-pair term out
                const double ac = static_cast<double>(self_clamped_coef(TENSOR, k.clampv, k.k2));
                vx = fin.mu0 * static_cast<double>(f.x) + fin.c1 * (vx - ac * static_cast<double>(f.x));
                vy = fin.mu0 * static_cast<double>(f.y) + fin.c1 * (vy - ac * static_cast<double>(f.y));
                vz = fin.mu0 * static_cast<double>(f.z) + fin.c1 * (vz - ac * static_cast<double>(f.z));
                fin.vel[i_mine] = make_float4(static_cast<float>(vx), static_cast<float>(vy),
                                              static_cast<float>(vz), 0.f);
                if (fin.mode != FIN_VEL) {
                    const float4 ph = fin.pos_base[i_mine];
                    double X = ph.x, Y = ph.y, Z = ph.z;
                    if (fin.pos_comp) {
                        const float4 pl = fin.pos_lo[i_mine];
                        X += pl.x, Y += pl.y, Z += pl.z;
                    }
                    const double h = (fin.mode == FIN_HALF) ? 0.5 * fin.dt : fin.dt;
                    X += h * vx, Y += h * vy, Z += h * vz;
                    const float xh = static_cast<float>(X), yh = static_cast<float>(Y), zh = static_cast<float>(Z);
                    fin.pos_out[i_mine] = make_float4(xh, yh, zh, 0.f);
                    if (fin.mode != FIN_HALF)
                        fin.pos_lo[i_mine] =
                            fin.pos_comp ? make_float4(static_cast<float>(X - static_cast<double>(xh)),
                                                       static_cast<float>(Y - static_cast<double>(yh)),
                                                       static_cast<float>(Z - static_cast<double>(zh)), 0.f)
                                         : make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
        }
        __syncthreads();  // `red` and `s_last` are reused by the next segment
        if (u == u_begin) SD_WTRACE(5);
        u += nt;
    }
    SD_WTRACE(6);
}

}  // namespace sd
