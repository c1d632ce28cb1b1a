// sd_common.cuh -- shared device helpers of libsd_b200: mbarrier / bulk-copy (TMA) wrappers,
// the static work schedule and the packed-particle record layout.
//
// Data layout in HBM (all context-owned):
//   rec32 : [Nrec][2] float4  = { x, y, z, 0 | c1 Fx, c1 Fy, c1 Fz, 0 }  one 32-byte record per
//           particle (c1 = mu0 3a/4 folded into the force, see PairCoefT below),
//   rec64 : [Nrec][2] double4 = same in fp64 (64 bytes),
//           the paper's "32 bytes per particle (2 x float4)" record.  Nrec is N
//           rounded up to SD_REC_ALIGN; pad records sit at SD_PAD_POS with zero force, so they
//           add exactly 0 to every sum and a j-tile is always one full bulk copy.  (With a
//           periodic box the wrapped image of a pad can land anywhere: it still adds 0 on the
//           fast path, and the exact body skips j >= N.)
//   part  : [slot][Nrec][2]   = compensated partial sums (hi, lo) of one (i-block, j-range)
//           segment; combined by the finalize kernel.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define SD_REC_ALIGN 2048        // Nrec granularity (>= largest i-block and j-tile)
#define SD_PAD_POS 1.0e15f       // pad-record coordinate: r^2 ~ 3e30 stays finite in fp32
#define SD_DUMMY_I_POS (-1.0e15f) // coordinate given to i-lanes beyond N

namespace sd {

// ---- mbarrier + 1-D bulk async copy (cp.async.bulk -> SASS UBLKCP) --------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// global -> shared bulk copy of `bytes` (multiple of 16, 16-byte aligned both sides); completion
// is signalled on `bar` as a transaction count.
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, uint32_t bytes,
                                          uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(smem_dst)),
        "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// ---- static schedule ("stream-K" over the flattened (i-block, j-tile) grid) ------------------
// Unit u = b * T + t  (b: i-block, t: j-tile).  CTA c owns units [cta_u0[c], cta_u0[c+1]).  The
// pieces of that range that fall into one i-block are "segments"; segment (c, b) writes its
// partial sums to slot c - blk_first_cta[b] of block b.  Everything is computed on the host in
// sd_create and is deterministic: no atomics, bit-reproducible results.
struct Schedule {
    const long long* cta_u0;   // [G + 1]
    const int* blk_first_cta;  // [B]
    const int* blk_nslots;     // [B]
    const int* cta_piece;      // [G] piece (index into cta_u0) of CTA blockIdx.x, see sd_b200.cu
    int T;                     // j-tiles
    int B;                     // i-blocks
    int G;                     // CTAs
};

// Coefficients of the pair kernels in "folded" units: the force lane of a record holds
// F' = c1 F with c1 = mu0 3a/4 (the 1/r coefficient of Eq. 4 / 7b), so that
//   far field  T.F = (1/r + k2/r^3) F' + (1 - 3 k2/r^2)/r^3 (d.F') d ,   k2 = (a^3/2)/(3a/4) = 2a^2/3
//   overlap    T.F = (mu0r + ovA r) F' + (ovB/r) (d.F') d                (A4)
// and every coefficient depends on a only.
template <typename S>
struct PairCoefT {
    S k2;     // 2 a^2 / 3
    S m3k2;   // -2 a^2
    S mu0r;   // mu0 / c1 = 4 / (3a)      (coincident centres; self term in the finalize kernel)
    S ovA;    // -3 / (8 a^2)             overlap branch: A = mu0r + ovA * r
    S ovB;    // 1 / (8 a^2)              overlap branch: B = ovB / r
    S thr;    // careful-pass threshold on r^2: 4a^2 for RPY, tiny for Oseen (only r == 0)
    S clampv; // 4 a^2: lower clamp of r^2 in the careful pass (both tensors)
    // periodic cube of side L, nearest image only (PAPER.md:115 footnote 1); unused in free space
    S invL;   // 1 / L rounded to S
    S mL;     // -L
    S magic;  // 1.5 * 2^23 (float) / 1.5 * 2^52 (double): fma(d, invL, magic) - magic = rint(d invL)
};
typedef PairCoefT<float> PairCoef;
typedef PairCoefT<double> PairCoef64;

}  // namespace sd
