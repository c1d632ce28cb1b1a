// sd_pairs_f32.cuh -- all-pairs mobility kernel, fp32 terms with compensated accumulation.
//
// Computes, for every particle i of the CTA's i-blocks and every j of its j-range,
//     t_ij = A(r) F_j + B(r) (d.F_j) d ,   d = r_i - r_j                (Eq. 7a/7b)
// without ever forming the 3x3 tensor, and writes compensated partial sums.
//
// Mapping (B200-first, differs from the paper's Alg. 1/2):
//  * one thread owns I = 2*I2 particles i, held in registers as I2 packed f32x2 pairs; all FP32
//    work is issued as packed FFMA2/FMUL2/FADD2 (two i per instruction, the j operand is a
//    broadcast scalar), halving the issue slots per pair interaction;
//  * j data (32-byte records) are staged in shared memory by 1-D bulk async copies
//    (cp.async.bulk + mbarrier transaction counts) in a kStages-deep ring; every lane reads the
//    same record (LDS.128 broadcast), so there are no bank conflicts by construction;
//  * the 1/r coefficient c1 = mu0 3a/4 is folded into the force lane of the records
//    (F' = c1 F, written by the pack / finalize kernels), so the far-field tensor becomes
//        T(d).F = A' F' + B' (d.F') d ,  A' = 1/r + k2/r^3 ,  B' = (1 - 3 k2/r^2)/r^3 ,
//    k2 = c2/c1 = 2a^2/3: the coefficients depend on a only and cost 5 packed instructions;
//  * 1/r and 1/r^2 come from MUFU.RSQ and MUFU.RCP (two MUFU issue as cheaply as the packed
//    multiply they replace); everything else is FMUL2/FFMA2/FADD2: 20 packed FP32 instructions
//    per two pairs (Rotne-Prager), 17 (Oseen);
//  * accumulation (terms of very different magnitude): plain fp32 adds inside a
//    chunk of kChunk consecutive j, Kahan merge of the chunk sum into (s, c) per particle;
//  * the r < 2a branch and the j == i exclusion are NOT evaluated per pair: the fast body
//    evaluates the far-field formula unconditionally and tracks min r^2 per chunk; a chunk
//    with min r^2 < 4a^2 (an overlapping pair, or the self pair r = 0) is discarded and redone
//    by the exact, branching slow body.  Overlaps are rare (about 8 phi neighbours per
//    particle), the self pair occurs once per row.
#pragma once
#include "sd_common.cuh"

namespace sd {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kTJ = 128;     // j records per tile (4 KiB)
// Second tile size of the 2-particle-per-thread variant: 32 records, i.e. four times the work
// units, for a finer balance over the 444 resident CTAs.  Measured per product with the SM-balanced
// piece map against 128-record tiles: 3-10 % faster for 4500 <= N <= 11000 (N = 6000: 61.6 -> 55.4
// us), equal at 4000 and 12288, 20 % slower at N <= 3000 (30.8 -> 36.9 us: four times the slots to
// reduce, a tile hand-over every 32 j), 1.6 % slower at 14000.  Used for kTJSmallMinN <= N <= kTJSmallMaxN.
constexpr int kTJSmall = 32;
// Third tile size, 256 records (8 KiB), for the 8-particle-per-thread kernel at N >= kRepairMaxN: a tile
// hand-over (empty-barrier arrival, the next bulk copy issued by thread 0, full-barrier wait, restart of
// the j pipeline) costs about 330 cycles of the CTA's slowest warp -- 1.2 % of a 128-record tile.
// Measured (same box, same process, L2 flushed): N = 1 M 0.6602 -> 0.6647 of the roofline, 262 144
// 0.6576 -> 0.6622; 32-record tiles: -1.1 ... -3.7 % at 32 768 ... 131 072.  Below kRepairMaxN the coarser
// units cost in balance what the hand-overs save (65 536: -0.7 %, 131 072: +0.1 %); 512-record tiles need
// dynamic shared memory, and addressing the ring through a pointer instead of the static array moved the
// hot loop's register allocation (-1.7 % at every size).
constexpr int kTJLarge = 256;
constexpr int kTJSmallMinN = 4300;
constexpr int kTJSmallMaxN = 12288;
constexpr int kStages = 4;   // ring depth
constexpr int kPrefetch = 2; // tiles in flight ahead of the one being consumed
constexpr int kChunk = 32;   // j per compensation chunk
constexpr int kUnrollJ = 4;  // j per unrolled loop body (2: -3 %, 8: -2.7 % at N = 1 M)
// measured crossovers of the particles-per-thread variants (profiles/r01e_sweep.md)
constexpr int kIpt4Min = 20480;    // above: 4 particles per thread in fp32
constexpr int kIpt4MinBox = 14336; // same in the periodic box (29 instead of 20 instructions per step)
constexpr int kIpt2Min64 = 12288;  // above: 2 particles per thread in fp64
constexpr int kIpt8Min = 29000;    // above: 8 per thread in fp32 (r01f: 30000: 717 against 730 us, 28000: 654 against 647)
constexpr int kIpt8MinBox = 43000; // same in the periodic box (36000: 1404 against 1370 us, 49152: 2433 against 2455)
constexpr int kIpt4Min64 = 40960;  // above: 4 per thread in fp64

enum { TENSOR_RPY = 0, TENSOR_OSEEN = 1 };
enum { ACC_KAHAN = 0, ACC_PLAIN = 1 };
// How the j records reach the threads (ablation of PAPER.md:111-241, Appendix A; sd_set_staging):
//   STAGE_BULK  bulk async copies (TMA engine) into a ring of shared-memory tiles, mbarriers only
//   STAGE_NAIVE no staging: every thread loads the record from global memory (one address per
//               warp, broadcast through L1), the paper's "naive" scheme (Alg. 1)
//   STAGE_SYNC  the CTA copies a tile into shared memory between two __syncthreads, the paper's
//               "tiling" scheme (Alg. 2 generalised from one warp to the whole block)
enum { STAGE_BULK = 0, STAGE_NAIVE = 1, STAGE_SYNC = 2 };

__device__ __forceinline__ float rsq_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// Packed f32x2 values live in one 64-bit register (an aligned register pair) and are only
// touched through these wrappers, so that ptxas keeps loop-invariant pairs packed instead of
// re-assembling them from two scalars before every use.  A pair built from the same scalar
// twice is folded by ptxas into the broadcast operand form (`R12.F32`) of FFMA2/FMUL2/FADD2.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f32x2 bc2(float s) { return pk2(s, s); }
__device__ __forceinline__ float lo2(f32x2 v) {
    float lo;
    asm("{\n.reg .b32 t;\nmov.b64 {%0, t}, %1;\n}" : "=f"(lo) : "l"(v));
    return lo;
}
__device__ __forceinline__ float hi2(f32x2 v) {
    float hi;
    asm("{\n.reg .b32 t;\nmov.b64 {t, %0}, %1;\n}" : "=f"(hi) : "l"(v));
    return hi;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// Far-field body for the I2 packed groups of a thread (2*I2 particles i) against one j, written
// stage by stage so that consecutive instructions share the broadcast j operand (operand-reuse
// cache): the register-file read ports, not the FMA pipe, are the binding resource (an FFMA2
// with three distinct register operands in one bank takes 3 cycles instead of 2).
// 20 packed FP32 instructions + 4 MUFU per two pairs for Rotne-Prager, 17 + 4 for Oseen.
// fj holds F' = c1 F (see the file header); k.k2 = 2a^2/3, k.m3k2 = -2a^2.
// PBC (periodic cube, nearest image only; PAPER.md:115 footnote 1): every component of d is
// replaced by d - L n with n = rint(d / L) taken as (fma(d, 1/L, M) - M), M = 1.5 * 2^23: the
// fma rounds the exact product d * fl(1/L) to an integer, ties to even (reading B2).
// 3 more packed instructions per component: 29 per two pairs (Rotne-Prager), 26 (Oseen).
// CLAMP (the "careful" pass, see the kernel): r^2 is clamped from below to k.clampv = 4a^2
// before the MUFUs, so that every pair -- the self pair and overlapping pairs included -- adds a
// finite term of ordinary magnitude; the unclamped r^2 of every pair is returned in r2out and
// the caller corrects the few pairs below the clamp.  Branch-free, 2 FMNMX per two pairs more.
// MNG: min r^2 is tracked per packed group in mng[m] instead of in the single mn (same number of
// instructions; the warp-split kernel repairs only the groups that met a close pair).
template <int I2, int TENSOR, bool PBC, bool CLAMP, bool MNG = false>
__device__ __forceinline__ void pair_fast_staged(const f32x2 (&xi)[I2], const f32x2 (&yi)[I2],
                                                 const f32x2 (&zi)[I2], const float4 pj,
                                                 const float4 fj, const PairCoef& k,
                                                 f32x2 (&px)[I2], f32x2 (&py)[I2], f32x2 (&pz)[I2],
                                                 float& mn, float (&r2out)[2 * I2], float* mng = nullptr) {
    f32x2 dx[I2], dy[I2], dz[I2], r2[I2], inv[I2], inv2[I2], dF[I2], A[I2], Bd[I2];
    const f32x2 xj = bc2(pj.x), yj = bc2(pj.y), zj = bc2(pj.z);
    const f32x2 fx = bc2(fj.x), fy = bc2(fj.y), fz = bc2(fj.z);
#pragma unroll
    for (int m = 0; m < I2; ++m) dx[m] = sub2(xi[m], xj);
#pragma unroll
    for (int m = 0; m < I2; ++m) dy[m] = sub2(yi[m], yj);
#pragma unroll
    for (int m = 0; m < I2; ++m) dz[m] = sub2(zi[m], zj);
    if (PBC) {
        const f32x2 il = bc2(k.invL), mg = bc2(k.magic), nl = bc2(k.mL);
#pragma unroll
        for (int m = 0; m < I2; ++m) {
            const f32x2 qx = sub2(fma2(dx[m], il, mg), mg);
            const f32x2 qy = sub2(fma2(dy[m], il, mg), mg);
            const f32x2 qz = sub2(fma2(dz[m], il, mg), mg);
            dx[m] = fma2(qx, nl, dx[m]);
            dy[m] = fma2(qy, nl, dy[m]);
            dz[m] = fma2(qz, nl, dz[m]);
        }
    }
#pragma unroll
    for (int m = 0; m < I2; ++m) {
        r2[m] = mul2(dx[m], dx[m]);
        r2[m] = fma2(dy[m], dy[m], r2[m]);
        r2[m] = fma2(dz[m], dz[m], r2[m]);
    }
#pragma unroll
    for (int m = 0; m < I2; ++m) {
        float a = lo2(r2[m]), b = hi2(r2[m]);
        if (CLAMP) {
            r2out[2 * m] = a;
            r2out[2 * m + 1] = b;
            a = fmaxf(a, k.clampv);
            b = fmaxf(b, k.clampv);
        } else {
            if (MNG) mng[m] = fminf(mng[m], fminf(a, b));
            else mn = fminf(mn, fminf(a, b));
        }
        inv[m] = pk2(rsq_approx(a), rsq_approx(b));
        inv2[m] = pk2(rcp_approx(a), rcp_approx(b));
    }
#pragma unroll
    for (int m = 0; m < I2; ++m) dF[m] = mul2(dx[m], fx);
#pragma unroll
    for (int m = 0; m < I2; ++m) dF[m] = fma2(dy[m], fy, dF[m]);
#pragma unroll
    for (int m = 0; m < I2; ++m) dF[m] = fma2(dz[m], fz, dF[m]);
#pragma unroll
    for (int m = 0; m < I2; ++m) {
        const f32x2 inv3 = mul2(inv[m], inv2[m]);
        if (TENSOR == TENSOR_RPY) {
            A[m] = fma2(inv3, bc2(k.k2), inv[m]);                          // 1/r + k2/r^3
            const f32x2 g = mul2(inv3, dF[m]);                             // (d.F')/r^3
            const f32x2 Q = fma2(inv2[m], bc2(k.m3k2), bc2(1.0f));         // 1 - 3 k2/r^2
            Bd[m] = mul2(g, Q);                                            // B' (d.F')
        } else {
            A[m] = inv[m];                                                 // 1/r
            Bd[m] = mul2(inv3, dF[m]);                                     // (d.F')/r^3
        }
    }
#pragma unroll
    for (int m = 0; m < I2; ++m) px[m] = fma2(A[m], fx, px[m]);
#pragma unroll
    for (int m = 0; m < I2; ++m) py[m] = fma2(A[m], fy, py[m]);
#pragma unroll
    for (int m = 0; m < I2; ++m) pz[m] = fma2(A[m], fz, pz[m]);
#pragma unroll
    for (int m = 0; m < I2; ++m) {
        px[m] = fma2(Bd[m], dx[m], px[m]);
        py[m] = fma2(Bd[m], dy[m], py[m]);
        pz[m] = fma2(Bd[m], dz[m], pz[m]);
    }
}

// Exact body for one (i, j): self exclusion, coincident centres, overlap branch (A4,
// A5), in the same folded units as the fast body (fj = c1 F_j, coefficients relative to c1).
template <int TENSOR, bool PBC>
__device__ __forceinline__ void pair_exact(const float xi, const float yi, const float zi,
                                           const bool self, const float4 pj, const float4 fj,
                                           const PairCoef& k, float& px, float& py, float& pz) {
    if (self) return;
    float dx = xi - pj.x, dy = yi - pj.y, dz = zi - pj.z;
    if (PBC) {  // same nearest-image rule as the fast body
        dx = __fmaf_rn(__fsub_rn(__fmaf_rn(dx, k.invL, k.magic), k.magic), k.mL, dx);
        dy = __fmaf_rn(__fsub_rn(__fmaf_rn(dy, k.invL, k.magic), k.magic), k.mL, dy);
        dz = __fmaf_rn(__fsub_rn(__fmaf_rn(dz, k.invL, k.magic), k.magic), k.mL, dz);
    }
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (r2 == 0.0f) {
        if (TENSOR == TENSOR_RPY) {  // limit of the overlap branch: mu0 F_j
            px = fmaf(k.mu0r, fj.x, px);
            py = fmaf(k.mu0r, fj.y, py);
            pz = fmaf(k.mu0r, fj.z, pz);
        }
        return;
    }
    const float inv = rsq_approx(r2);
    const float dF = fmaf(dz, fj.z, fmaf(dy, fj.y, dx * fj.x));
    float A, B;
    if (TENSOR == TENSOR_RPY) {
        if (r2 < k.thr) {  // r < 2a
            const float r = r2 * inv;
            A = fmaf(k.ovA, r, k.mu0r);
            B = k.ovB * inv;
        } else {
            const float inv2 = inv * inv;
            const float inv3 = inv2 * inv;
            A = fmaf(k.k2, inv3, inv);
            B = fmaf(k.m3k2, inv2, 1.0f) * inv3;
        }
    } else {
        A = inv;
        B = inv * inv * inv;
    }
    const float Bd = B * dF;
    px = fmaf(A, fj.x, px);
    py = fmaf(A, fj.y, py);
    pz = fmaf(A, fj.z, pz);
    px = fmaf(Bd, dx, px);
    py = fmaf(Bd, dy, py);
    pz = fmaf(Bd, dz, pz);
}

// What the CLAMP body added for one (i, j) whose r^2 lies below the clamp: the far-field formula
// evaluated with 1/r := 1/sqrt(clampv) on the true d.  Subtracted again by the careful pass (and
// replaced by pair_exact unless the pair is the self pair).  d = 0 for the self pair: A_c F' only.
template <int TENSOR, bool PBC>
__device__ __forceinline__ void pair_clamped_sub(const float xi, const float yi, const float zi,
                                                 const float4 pj, const float4 fj,
                                                 const PairCoef& k, float& px, float& py,
                                                 float& pz) {
    float dx = xi - pj.x, dy = yi - pj.y, dz = zi - pj.z;
    if (PBC) {
        dx = __fmaf_rn(__fsub_rn(__fmaf_rn(dx, k.invL, k.magic), k.magic), k.mL, dx);
        dy = __fmaf_rn(__fsub_rn(__fmaf_rn(dy, k.invL, k.magic), k.magic), k.mL, dy);
        dz = __fmaf_rn(__fsub_rn(__fmaf_rn(dz, k.invL, k.magic), k.magic), k.mL, dz);
    }
    const float inv = rsq_approx(k.clampv), inv2 = rcp_approx(k.clampv);
    const float inv3 = inv * inv2;
    const float dF = fmaf(dz, fj.z, fmaf(dy, fj.y, dx * fj.x));
    float A, Bd;
    if (TENSOR == TENSOR_RPY) {
        A = fmaf(inv3, k.k2, inv);
        Bd = (inv3 * dF) * fmaf(inv2, k.m3k2, 1.0f);
    } else {
        A = inv;
        Bd = inv3 * dF;
    }
    px = fmaf(-A, fj.x, px);
    py = fmaf(-A, fj.y, py);
    pz = fmaf(-A, fj.z, pz);
    px = fmaf(-Bd, dx, px);
    py = fmaf(-Bd, dy, py);
    pz = fmaf(-Bd, dz, pz);
}

// Coefficient of F'_i in the term the CLAMP body adds for the self pair (d = 0, r^2 clamped to
// k.clampv): A_c = 1/r_c + k2/r_c^3 (Rotne-Prager) or 1/r_c (Oseen), formed by the very
// instructions of pair_fast_staged so that the finalize kernel subtracts what the pair kernel
// added.  The d-dependent part of the term is exactly 0.
__device__ __forceinline__ float self_clamped_coef(const int tensor, const float clampv, const float k2) {
    const float inv = rsq_approx(clampv), inv2 = rcp_approx(clampv);
    const float inv3 = __fmul_rn(inv, inv2);
    return tensor == TENSOR_RPY ? __fmaf_rn(inv3, k2, inv) : inv;
}

// Repair of one chunk whose packed pass met a pair below the clamp (overlapping spheres,
// coincident centres).  The unclamped body has then added a far-field term of enormous size to the
// sum of ONE particle; the other packed groups of the lane are fine.  Only the groups flagged in
// kernel's `groups` mask are redone, one call of chunk_fix_group each: the chunk sum restarts from
// its base (0, or the running sum at chunk start without compensation), every pair goes through the
// clamped packed body for that one group (finite terms of ordinary size), and the pairs below the
// clamp are put right one by one -- clamped term out, exact term in.  About a quarter of an
// ordinary chunk pass per flagged group, where redoing the chunk for all groups with per-pair
// checks cost six to eight passes (at phi = 0.01 one chunk pass in 6 is hit at N = 4096, one in 50
// at N = 32768: the mid-N loss of round 1).
//   cp / cf : positions / forces of the chunk's records, JS float4 apart from one j to the next
//   ISTEP   : index distance between the particles of consecutive slots (m, half) of a lane
// Convention kept for the epilogue: a self pair leaves the clamped term A_c F'_i in the sum.
// It is a real call (__noinline__, operands by value): inlined into the kernel it took part in the
// register allocation of the hot loop (22 accumulator copies per 4 j in the warp-split kernel,
// -2 % in the classic one); as a call the hot loop does not know it exists.
struct P3 {
    f32x2 x, y, z;
};
template <int TENSOR, bool PBC, int JS, int ISTEP>
__device__ __noinline__ P3 chunk_fix_group(const f32x2 x, const f32x2 y, const f32x2 z, const float4* cp,
                                           const float4* cf, const int j0, const int len, const int N,
                                           const int i0, const PairCoef k, const P3 base) {
    f32x2 x1[1] = {x}, y1[1] = {y}, z1[1] = {z};
    f32x2 p1x[1] = {base.x}, p1y[1] = {base.y}, p1z[1] = {base.z};
    const float xa = lo2(x), ya = lo2(y), za = lo2(z);
    const float xb = hi2(x), yb = hi2(y), zb = hi2(z);
    float mnd = 0.f, r2p[2];
#pragma unroll 2
    for (int jj = 0; jj < len; ++jj) {
        const float4 pj = cp[jj * JS];
        const float4 fj = cf[jj * JS];
        const int j = j0 + jj;
        pair_fast_staged<1, TENSOR, PBC, true>(x1, y1, z1, pj, fj, k, p1x, p1y, p1z, mnd, r2p);
        const bool fix0 = r2p[0] < k.clampv && j != i0;
        const bool fix1 = r2p[1] < k.clampv && j != i0 + ISTEP;
        if ((fix0 || fix1) && j < N) {
            float ax = lo2(p1x[0]), ay = lo2(p1y[0]), az = lo2(p1z[0]);
            float bx = hi2(p1x[0]), by = hi2(p1y[0]), bz = hi2(p1z[0]);
            if (fix0) {
                pair_clamped_sub<TENSOR, PBC>(xa, ya, za, pj, fj, k, ax, ay, az);
                pair_exact<TENSOR, PBC>(xa, ya, za, false, pj, fj, k, ax, ay, az);
            }
            if (fix1) {
                pair_clamped_sub<TENSOR, PBC>(xb, yb, zb, pj, fj, k, bx, by, bz);
                pair_exact<TENSOR, PBC>(xb, yb, zb, false, pj, fj, k, bx, by, bz);
            }
            p1x[0] = pk2(ax, bx);
            p1y[0] = pk2(ay, by);
            p1z[0] = pk2(az, bz);
        }
    }
    P3 r;
    r.x = p1x[0], r.y = p1y[0], r.z = p1z[0];
    return r;
}

__device__ __forceinline__ void kahan_merge2(f32x2& s, f32x2& c, const f32x2 p) {
    const f32x2 y = sub2(p, c);
    const f32x2 t = add2(s, y);
    c = sub2(sub2(t, s), y);
    s = t;
}

// REPAIR: what happens to a chunk that holds a pair below the clamp (or the warp's self pairs).
//   0  round-1 careful pass: the whole chunk again through the clamped body with per-pair checks
//      (six to eight chunk passes; its code shares the kernel's register allocation)
//   1  diagonal chunks branch-free, flagged packed groups repaired by a call of chunk_fix_group
// Measured (profiles/r02_mid_n.md): 1 is 5 % faster at N = 32 768, 1.6 % at 65 536, equal at 131 072
// and 0.9 % SLOWER at N = 1 048 576 (the FFMA2 loop is the same text, its registers are not), so the
// dispatcher takes 1 below kRepairMaxN and 0 above.
constexpr int kRepairMaxN = 200000;
template <int I2, int TENSOR, int ACC, bool PBC, int STAGE = STAGE_BULK, int TJ = kTJ, int REPAIR = 1>
__global__ void __launch_bounds__(kThreads, (I2 == 1) ? 3 : ((I2 == 2) ? 2 : 1))
pairs_f32_kernel(const float4* __restrict__ rec, float4* __restrict__ part, const Schedule sch,
                 const PairCoef k, const int N, const long long slot_stride) {
    constexpr int I = 2 * I2;
    constexpr int IB = kThreads * I;
    static_assert(TJ % kChunk == 0, "a tile is a whole number of compensation chunks");
    __shared__ __align__(128) float4 tiles[kStages][TJ * 2];
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

    // producer state (thread 0): next unit to fetch and its j-tile index
    int pf_n = 0;
    int pf_t = static_cast<int>(u_begin % T);
    auto produce = [&]() {
        const int s = pf_n % kStages;
        const int q = pf_n / kStages;
        if (q > 0) mbar_wait(&empty_bar[s], (q - 1) & 1);
        mbar_arrive_expect_tx(&full_bar[s], TJ * 32);
        bulk_load(&tiles[s][0], rec + static_cast<size_t>(pf_t) * (TJ * 2), TJ * 32, &full_bar[s]);
        ++pf_n;
        if (++pf_t == T) pf_t = 0;
    };
    if (tid == 0) {
        for (int q = 0; STAGE == STAGE_BULK && q < kPrefetch && pf_n < n_units; ++q) produce();
    }

    int n = 0;  // tiles consumed so far by this CTA
    long long u = u_begin;
    while (u < u_end) {
        const int b = static_cast<int>(u / T);
        const int t0 = static_cast<int>(u - static_cast<long long>(b) * T);
        const long long left = u_end - u;
        const int nt = (left < static_cast<long long>(T - t0)) ? static_cast<int>(left) : (T - t0);
        const int i_first = b * IB + tid;  // particle of (m = 0, half 0)

        f32x2 xi[I2], yi[I2], zi[I2];

#pragma unroll
        for (int m = 0; m < I2; ++m) {
            const int i0 = i_first + (2 * m) * kThreads;
            const int i1 = i0 + kThreads;
            const float4 d = make_float4(SD_DUMMY_I_POS, SD_DUMMY_I_POS, SD_DUMMY_I_POS, 0.f);
            const float4 p0 = (i0 < N) ? rec[2 * static_cast<size_t>(i0)] : d;
            const float4 p1 = (i1 < N) ? rec[2 * static_cast<size_t>(i1)] : d;
            // x + 0 through a packed add: the result is born as an aligned register pair (a
            // bare pack of two LDG.128 lanes makes ptxas re-assemble the pair at every use)
            const f32x2 zero = bc2(0.f);
            xi[m] = add2(pk2(p0.x, p1.x), zero);
            yi[m] = add2(pk2(p0.y, p1.y), zero);
            zi[m] = add2(pk2(p0.z, p1.z), zero);
        }
        f32x2 sx[I2], sy[I2], sz[I2], cx[I2], cy[I2], cz[I2];  // Kahan (sum, compensation)
        f32x2 px[I2], py[I2], pz[I2];                          // chunk sum (PLAIN: running sum)
#pragma unroll
        for (int m = 0; m < I2; ++m) {
            sx[m] = sy[m] = sz[m] = cx[m] = cy[m] = cz[m] = bc2(0.f);
            px[m] = py[m] = pz[m] = bc2(0.f);
        }

        for (int tt = 0; tt < nt; ++tt, ++n) {
            const int s = n % kStages;
            const float4* tile;
            if (STAGE == STAGE_BULK) {
                if (tid == 0 && pf_n < n_units) produce();
                mbar_wait(&full_bar[s], (n / kStages) & 1);
                tile = &tiles[s][0];
            } else if (STAGE == STAGE_NAIVE) {
                tile = rec + static_cast<size_t>(t0 + tt) * (TJ * 2);
            } else {
                __syncthreads();  // everybody is done with the previous tile
                for (int q = tid; q < TJ * 2; q += kThreads) tiles[0][q] = rec[static_cast<size_t>(t0 + tt) * (TJ * 2) + q];
                __syncthreads();
                tile = &tiles[0][0];
            }
            const int jbase = (t0 + tt) * TJ;

#pragma unroll 1
            for (int ch = 0; ch < TJ / kChunk; ++ch) {
                const float4* cj = tile + ch * (kChunk * 2);
                f32x2 qx[I2], qy[I2], qz[I2];  // value of p at chunk start (PLAIN only)
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
                if (REPAIR == 0) {
                    float mn = 3.0e38f;
                    float r2v[2 * I2];
                    const int j0 = jbase + ch * kChunk;
                    // the chunk that holds this warp's own particles (self pairs, r = 0)
                    const int rel = j0 - (i_first - lane);
                    const bool diag = rel >= 0 && (rel % kThreads) == 0 && rel < I * kThreads;
                    if (!diag) {
    #pragma unroll kUnrollJ
                        for (int jj = 0; jj < kChunk; ++jj) {
                            const float4 pj = cj[2 * jj];
                            const float4 fj = cj[2 * jj + 1];
                            pair_fast_staged<I2, TENSOR, PBC, false>(xi, yi, zi, pj, fj, k, px, py, pz,
                                                                     mn, r2v);
                        }
                    }
                    if (diag || mn < k.thr) {
                        // careful pass: self pairs, overlapping pairs or coincident centres sit in this
                        // chunk.  Every pair goes through the clamped packed body (finite terms of
                        // ordinary size, so nothing cancels); the pairs below the clamp are then put
                        // right one by one: clamped term out, exact term (none for the self pair) in.
                        // (The cheaper repair of the warp-split kernel, chunk_fix, was measured here too:
                        // it moves the register allocation of the hot loop, -2.0 % at N = 1 M, -1.4 % at
                        // 65 536, +0.9 % at 32 768; profiles/r02_mid_n.md.)
    #pragma unroll
                        for (int m = 0; m < I2; ++m) {
                            if (ACC == ACC_KAHAN) {
                                px[m] = py[m] = pz[m] = bc2(0.f);
                            } else {
                                px[m] = qx[m];
                                py[m] = qy[m];
                                pz[m] = qz[m];
                            }
                        }
    #pragma unroll 2
                        for (int jj = 0; jj < kChunk; ++jj) {
                            const float4 pj = cj[2 * jj];
                            const float4 fj = cj[2 * jj + 1];
                            const int j = j0 + jj;
                            pair_fast_staged<I2, TENSOR, PBC, true>(xi, yi, zi, pj, fj, k, px, py, pz,
                                                                    mn, r2v);
    #pragma unroll
                            for (int m = 0; m < I2; ++m) {
                                // the self pair keeps its clamped term A_c F'_i: the finalize kernel
                                // takes it out again (self_clamped_coef), all rows at once, instead of
                                // 32 lanes walking through this branch one after the other
                                const int i0 = i_first + (2 * m) * kThreads;
                                const bool fix0 = r2v[2 * m] < k.clampv && j != i0;
                                const bool fix1 = r2v[2 * m + 1] < k.clampv && j != i0 + kThreads;
                                if ((fix0 || fix1) && j < N) {
                                    float ax = lo2(px[m]), ay = lo2(py[m]), az = lo2(pz[m]);
                                    float bx = hi2(px[m]), by = hi2(py[m]), bz = hi2(pz[m]);
                                    if (fix0) {
                                        pair_clamped_sub<TENSOR, PBC>(lo2(xi[m]), lo2(yi[m]), lo2(zi[m]),
                                                                      pj, fj, k, ax, ay, az);
                                        pair_exact<TENSOR, PBC>(lo2(xi[m]), lo2(yi[m]), lo2(zi[m]),
                                                                false, pj, fj, k, ax, ay, az);
                                    }
                                    if (fix1) {
                                        pair_clamped_sub<TENSOR, PBC>(hi2(xi[m]), hi2(yi[m]), hi2(zi[m]),
                                                                      pj, fj, k, bx, by, bz);
                                        pair_exact<TENSOR, PBC>(hi2(xi[m]), hi2(yi[m]), hi2(zi[m]),
                                                                false, pj, fj, k, bx, by, bz);
                                    }
                                    px[m] = pk2(ax, bx);
                                    py[m] = pk2(ay, by);
                                    pz[m] = pk2(az, bz);
                                }
                            }
                        }
                    }
                } else {
                    float mn = 3.0e38f;
                    float mng[I2];
    #pragma unroll
                    for (int m = 0; m < I2; ++m) mng[m] = 3.0e38f;
                    float r2v[2 * I2];
                    const int j0 = jbase + ch * kChunk;
                    // the chunk that holds this warp's own particles (self pairs, r = 0)
                    const int rel = j0 - (i_first - lane);
                    const bool diag = rel >= 0 && (rel % kThreads) == 0 && rel < I * kThreads;
                    unsigned groups = 0u;
                    if (!diag) {
    #pragma unroll kUnrollJ
                        for (int jj = 0; jj < kChunk; ++jj) {
                            const float4 pj = cj[2 * jj];
                            const float4 fj = cj[2 * jj + 1];
                            pair_fast_staged<I2, TENSOR, PBC, false, true>(xi, yi, zi, pj, fj, k, px, py, pz,
                                                                           mn, r2v, mng);
                        }
    #pragma unroll
                        for (int m = 0; m < I2; ++m) groups |= (mng[m] < k.thr ? 1u : 0u) << m;
                    } else {
                        int zeros = 0;
    #pragma unroll kUnrollJ
                        for (int jj = 0; jj < kChunk; ++jj) {
                            const float4 pj = cj[2 * jj];
                            const float4 fj = cj[2 * jj + 1];
                            pair_fast_staged<I2, TENSOR, PBC, true>(xi, yi, zi, pj, fj, k, px, py, pz, mn, r2v);
    #pragma unroll
                            for (int q = 0; q < I; ++q) {
                                const bool z = r2v[q] == 0.f;
                                zeros += z ? 1 : 0;
                                mng[q / 2] = fminf(mng[q / 2], z ? 3.0e38f : r2v[q]);
                            }
                        }
    #pragma unroll
                        for (int m = 0; m < I2; ++m) groups |= (mng[m] < k.clampv ? 1u : 0u) << m;
                        if (zeros != ((j0 + lane < N) ? 1 : 0)) groups = (1u << I2) - 1u;
                    }
                    if (groups) {
    #pragma unroll
                        for (int m = 0; m < I2; ++m) {
                            if ((groups >> m) & 1u) {
                                P3 base;
                                base.x = ACC == ACC_KAHAN ? bc2(0.f) : qx[m];
                                base.y = ACC == ACC_KAHAN ? bc2(0.f) : qy[m];
                                base.z = ACC == ACC_KAHAN ? bc2(0.f) : qz[m];
                                const P3 r = chunk_fix_group<TENSOR, PBC, 2, kThreads>(
                                    xi[m], yi[m], zi[m], cj, cj + 1, j0, kChunk, N, i_first + (2 * m) * kThreads, k, base);
                                px[m] = r.x, py[m] = r.y, pz[m] = r.z;
                            }
                        }
                    }
                }
                if (ACC == ACC_KAHAN) {
#pragma unroll
                    for (int m = 0; m < I2; ++m) {
                        kahan_merge2(sx[m], cx[m], px[m]);
                        kahan_merge2(sy[m], cy[m], py[m]);
                        kahan_merge2(sz[m], cz[m], pz[m]);
                    }
                }
            }
            if (STAGE == STAGE_BULK) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty_bar[s]);
            }
        }

        // partial sums of this segment: value = hi - lo
        const int slot = c - sch.blk_first_cta[b];
        float4* out = part + static_cast<size_t>(slot) * slot_stride * 2;
#pragma unroll
        for (int m = 0; m < I2; ++m) {
            const int i0 = i_first + (2 * m) * kThreads;
            const int i1 = i0 + kThreads;
            if (ACC == ACC_PLAIN) {
                sx[m] = px[m];
                sy[m] = py[m];
                sz[m] = pz[m];
            }
            if (i0 < N) {
                out[2 * static_cast<size_t>(i0)] =
                    make_float4(lo2(sx[m]), lo2(sy[m]), lo2(sz[m]), 0.f);
                out[2 * static_cast<size_t>(i0) + 1] =
                    make_float4(lo2(cx[m]), lo2(cy[m]), lo2(cz[m]), 0.f);
            }
            if (i1 < N) {
                out[2 * static_cast<size_t>(i1)] =
                    make_float4(hi2(sx[m]), hi2(sy[m]), hi2(sz[m]), 0.f);
                out[2 * static_cast<size_t>(i1) + 1] =
                    make_float4(hi2(cx[m]), hi2(cy[m]), hi2(cz[m]), 0.f);
            }
        }
        u += nt;
    }
}

}  // namespace sd
