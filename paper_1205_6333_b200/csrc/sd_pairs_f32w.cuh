// sd_pairs_f32w.cuh -- all-pairs mobility kernel, fp32, j split across the WARPS of a CTA, whole
// product in ONE launch (no pack kernel, no finalize kernel).
//
// Same pair arithmetic as sd_pairs_f32.cuh (packed FFMA2 body, chunked Kahan, clamped careful
// pass); what differs is the mapping, made for the under-filled regime N ~ 3e3 ... 1e5
// (PAPER.md:239, :273), where the classic kernel needs 2048-particle i-blocks to run its best
// inner loop and then has too few, too coarse work units for 148 SMs:
//  * all 8 warps of a CTA own the SAME 32 * 2 I2 particles i (8 per lane with I2 = 4, the inner
//    loop of the large-N kernel) and split every j tile between them: warp w takes the CH records
//    [w CH, (w + 1) CH) of each tile of TJ = 8 CH.  An i-block is 256 particles instead of 2048,
//    so N = 4096 already gives 16 x 32 units, and the per-unit tail (careful pass, diagonal tile)
//    shrinks by the same factor;
//  * the warps' compensated sums are combined through shared memory in fp64 in warp order, and
//    the CTA writes ONE (hi, lo) partial per particle and segment;
//  * the kernel reads the caller's pos / force arrays directly (two bulk copies per tile into a
//    tile laid out {TJ positions | TJ forces}; the ragged tail of the last tile comes from a
//    context-owned block of pad records), works in the folded units of sd_common.cuh on the RAW
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

constexpr int kWTJMax = 1024;  // largest tile of this kernel: size of the pad block halves
constexpr int kWMaxN = 6000;   // up to here the warp-split kernel runs by default (measured crossover)

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

template <int I2, int CH>
struct WShape {
    static constexpr int TJ = kWarps * CH;
    static constexpr int IBW = 64 * I2;  // particles per i-block: 32 lanes x 2 I2
    static constexpr size_t tile_bytes = static_cast<size_t>(kStages) * TJ * 2 * sizeof(float4);
    static constexpr size_t red_bytes = static_cast<size_t>(kWarps) * 6 * IBW * sizeof(float);
    static constexpr size_t smem_bytes = tile_bytes + red_bytes;
};

template <int I2, int TENSOR, int ACC, bool PBC, int CH>
__global__ void __launch_bounds__(kThreads, (I2 == 4) ? 1 : 2)
pairs_f32w_kernel(const float4* __restrict__ pos, const float4* __restrict__ frc,
                  const float4* __restrict__ padblk, float4* __restrict__ part,
                  int* __restrict__ blk_done, const Schedule sch, const PairCoef k, const FinArgs fin,
                  const int N, const long long slot_stride) {
    typedef WShape<I2, CH> W;
    constexpr int TJ = W::TJ;
    constexpr int IBW = W::IBW;
    constexpr int CK = CH < kChunk ? CH : kChunk;  // j per compensation chunk
    constexpr int NCH = CH / CK;                   // chunks per warp and tile
    static_assert(CK % kUnrollJ == 0 && CH % CK == 0 && TJ <= kWTJMax, "tile shape");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* tiles = reinterpret_cast<float4*>(smem_raw);                  // [kStages][2 TJ]
    float* red = reinterpret_cast<float*>(smem_raw + W::tile_bytes);      // [kWarps][6][IBW]
    __shared__ __align__(8) uint64_t full_bar[kStages];
    __shared__ __align__(8) uint64_t empty_bar[kStages];
    __shared__ int s_last;

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const int c = sch.cta_piece[blockIdx.x];
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
        float4* dst = tiles + static_cast<size_t>(s) * (2 * TJ);
        const int j0 = pf_t * TJ;
        const int valid = min(TJ, N - j0);
        mbar_arrive_expect_tx(&full_bar[s], TJ * 32);
        bulk_load(dst, pos + j0, valid * 16, &full_bar[s]);
        bulk_load(dst + TJ, frc + j0, valid * 16, &full_bar[s]);
        if (valid < TJ) {  // ragged tail: pad records (far away, zero force) complete the tile
            bulk_load(dst + valid, padblk, (TJ - valid) * 16, &full_bar[s]);
            bulk_load(dst + TJ + valid, padblk + kWTJMax, (TJ - valid) * 16, &full_bar[s]);
        }
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
        const int i_blk = b * IBW;
        const int i_first = i_blk + lane;  // particle of (m = 0, half 0); the others follow in steps of 32

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
        f32x2 sx[I2], sy[I2], sz[I2], cx[I2], cy[I2], cz[I2];
        f32x2 px[I2], py[I2], pz[I2];
#pragma unroll
        for (int m = 0; m < I2; ++m) {
            sx[m] = sy[m] = sz[m] = cx[m] = cy[m] = cz[m] = bc2(0.f);
            px[m] = py[m] = pz[m] = bc2(0.f);
        }

#pragma unroll 1
        for (int tt = 0; tt < nt; ++tt, ++n) {
            const int s = n % kStages;
            if (tid == 0 && pf_n < n_units) produce();
            mbar_wait(&full_bar[s], (n / kStages) & 1);
#pragma unroll 1
            for (int ch = 0; ch < NCH; ++ch) {
            // this warp's share of the tile: CH consecutive records = NCH compensation chunks
            const float4* cp = tiles + static_cast<size_t>(s) * (2 * TJ) + warp * CH + ch * CK;  // positions
            const float4* cf = cp + TJ;                                                          // forces
            const int j0 = (t0 + tt) * TJ + warp * CH + ch * CK;
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
            float mn = 3.0e38f;
            float r2v[2 * I2];
            // does this chunk hold self pairs (j = i) of the warp's particles?
            const bool diag = (j0 + CK > i_blk) && (j0 < i_blk + IBW);
            bool fix;
            if (!diag) {
#pragma unroll kUnrollJ
                for (int jj = 0; jj < CK; ++jj) {
                    const float4 pj = cp[jj];
                    const float4 fj = cf[jj];
                    pair_fast_staged<I2, TENSOR, PBC, false>(xi, yi, zi, pj, fj, k, px, py, pz, mn, r2v);
                }
                fix = mn < k.thr;
            } else {
                // diagonal chunk: the clamped body, branch-free (a self pair adds the finite term
                // A_c F'_i that the epilogue removes).  It is exact unless a pair other than the
                // self pairs lies below the clamp: min r^2 over the pairs with r^2 > 0, and the
                // number of exact zeros against the number of self pairs this lane meets here.
                int zeros = 0;
#pragma unroll kUnrollJ
                for (int jj = 0; jj < CK; ++jj) {
                    const float4 pj = cp[jj];
                    const float4 fj = cf[jj];
                    pair_fast_staged<I2, TENSOR, PBC, true>(xi, yi, zi, pj, fj, k, px, py, pz, mn, r2v);
#pragma unroll
                    for (int q = 0; q < 2 * I2; ++q) {
                        const bool z = r2v[q] == 0.f;
                        zeros += z ? 1 : 0;
                        mn = fminf(mn, z ? 3.0e38f : r2v[q]);
                    }
                }
                const int rel = j0 - i_blk;  // >= 0 here; this chunk holds the particles rel ... rel + CK - 1 of the block
                const int off = rel & 31;
                const bool mine = rel >= 0 && lane >= off && lane < off + CK && (i_first + (rel - off)) < N;
                fix = mn < k.clampv || zeros != (mine ? 1 : 0);
            }
            if (fix)  // rare: repair the sums of the particles that have a pair below the clamp here
                chunk_fix<I2, TENSOR, ACC, PBC, CK, 1, 32>(xi, yi, zi, cp, cf, j0, N, i_first, k,
                                                           diag ? k.clampv : k.thr, px, py, pz, qx, qy, qz);
            if (ACC == ACC_KAHAN) {
#pragma unroll
                for (int m = 0; m < I2; ++m) {
                    kahan_merge2(sx[m], cx[m], px[m]);
                    kahan_merge2(sy[m], cy[m], py[m]);
                    kahan_merge2(sz[m], cz[m], pz[m]);
                }
            }
            }  // chunks
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[s]);
        }

        // ---- combine the warps' sums (fp64, warp order): one (hi, lo) partial per particle ----
#pragma unroll
        for (int m = 0; m < I2; ++m) {
            if (ACC == ACC_PLAIN) {
                sx[m] = px[m];
                sy[m] = py[m];
                sz[m] = pz[m];
            }
            float* r0 = red + (warp * 6) * IBW + 64 * m + lane;  // [warp][component][particle]
            r0[0 * IBW] = lo2(sx[m]), r0[0 * IBW + 32] = hi2(sx[m]);
            r0[1 * IBW] = lo2(sy[m]), r0[1 * IBW + 32] = hi2(sy[m]);
            r0[2 * IBW] = lo2(sz[m]), r0[2 * IBW + 32] = hi2(sz[m]);
            r0[3 * IBW] = lo2(cx[m]), r0[3 * IBW + 32] = hi2(cx[m]);
            r0[4 * IBW] = lo2(cy[m]), r0[4 * IBW + 32] = hi2(cy[m]);
            r0[5 * IBW] = lo2(cz[m]), r0[5 * IBW + 32] = hi2(cz[m]);
        }
        __syncthreads();
        const int slot = c - sch.blk_first_cta[b];
        const int nslots = sch.blk_nslots[b];
        const int i_mine = i_blk + tid;  // the particle this thread reduces (tid < IBW)
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
        u += nt;
    }
}

}  // namespace sd
