// sd_lub.cuh -- lubrication correction of the forces.
//
//   mu0 f_sing(r_ij) = [ 1/(4 s) - (9/40) ln s ] rr^ - (1/6) ln s (I - rr^) ,  s = r_ij / a - 2   Eq. (8)
//   F_i <- F_i^ext - sum'_j f_sing(r_ij) . (v_i - v_j)         step 2 of the paper's loop
//
// with the velocities of the previous product and the primed sum over j != i with r_ij < 3a
// ("we truncate ad hoc at s = 1 or r = 3a").  The paper points to Verlet lists and particle
// reordering for this O(N) step; here it is a cell grid rebuilt on every
// call, no host synchronisation, deterministic:
//   lub_count_kernel    cell (3 ints, side >= 3a) and bucket (Morton code of the cell's low bits,
//                       H = 8^k >= N buckets) of every particle; bucket histogram by atomicAdd
//   lub_scan_*_kernel   exclusive scan of the H counters in two launches (block totals, then every
//                       block adds the totals before it to its own scan)
//   lub_scatter_kernel  particle indices into their buckets (atomic cursor), then
//   lub_sort_kernel     each bucket sorted by particle index: the summation order below, and
//                       with it every bit of the result, does not depend on the atomics
//   lub_gather_kernel   positions, velocities and cells copied into bucket order (the paper's
//                       "particle reordering"): neighbouring cells are neighbouring memory
//   lub_force_kernel    1 / 8 / 32 lanes per particle (by N), particles in bucket order: 27
//                       neighbour cells -> buckets -> candidates j (a candidate whose cell differs
//                       is a bucket alias and is skipped); the cut-off r^2 < 9a^2 is decided in
//                       the arithmetic of the context (fp32 fma chain in the fp32 modes,
//                       DESIGN.md reading C3), in fp32 contexts before any fp64 instruction; an
//                       accepted pair is evaluated in fp64 on the exact difference of the stored
//                       coordinates (s = r/a - 2 loses all digits in fp32 when the gap closes);
//                       sums in fp64 in a fixed order; writes F^ext - C rounded to the element type.
// Latency-bound (dependent loads bucket -> candidate -> position), 2 % of the HBM roofline at
// N = 1 M (profiles/r01d_lubrication.md).  Periodic box: cells = floor(L / 3a) per edge (>= 3
// required), neighbour cells wrap, displacements take the nearest image by the rule of the pair
// kernels.
#pragma once
#include "sd_common.cuh"
#include "sd_stream.cuh"

namespace sd {

constexpr double kLubSmin = 1.0e-3;  // lower clamp of s (reading C2: Eq. 8 diverges at contact)

struct LubGrid {
    double inv_cell;  // 1 / cell side
    double L, invL;   // periodic cube (0: free space)
    int nc;           // cells per edge in the box (0: free space, unbounded integer cells)
    unsigned mask;    // 2^bits - 1: low bits of a cell coordinate that enter the bucket index
};

// Bucket of a cell: Morton code of the low `bits` bits of its three coordinates (H = 2^(3 bits)
// buckets).  Neighbouring cells land in neighbouring buckets, so the 27 probes of a particle and
// the candidates they list are close in memory; cells 2^bits apart alias into one bucket and are
// told apart by the stored cell coordinates.
__device__ __forceinline__ unsigned lub_spread(unsigned v) {  // 10 bits -> every third bit
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
__device__ __forceinline__ unsigned lub_hash(int cx, int cy, int cz, unsigned mask) {
    return lub_spread(static_cast<unsigned>(cx) & mask) | (lub_spread(static_cast<unsigned>(cy) & mask) << 1) |
           (lub_spread(static_cast<unsigned>(cz) & mask) << 2);
}

__device__ __forceinline__ int lub_cell_coord(double x, const LubGrid& g) {
    if (g.nc > 0) {
        double u = x * g.invL;
        u -= floor(u);  // [0, 1)
        const int c = static_cast<int>(u * g.nc);
        return c < g.nc ? c : g.nc - 1;
    }
    return static_cast<int>(floor(x * g.inv_cell));
}

template <typename T4>
__global__ void __launch_bounds__(256)
lub_count_kernel(const T4* __restrict__ pos, int4* __restrict__ cell, unsigned* __restrict__ count,
                 const LubGrid g, const int N) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const T4 p = pos[i];
    const int cx = lub_cell_coord(p.x, g), cy = lub_cell_coord(p.y, g), cz = lub_cell_coord(p.z, g);
    const unsigned h = lub_hash(cx, cy, cz, g.mask);
    cell[i] = make_int4(cx, cy, cz, static_cast<int>(h));
    atomicAdd(&count[h], 1u);
}

__global__ void __launch_bounds__(256)
lub_scatter_kernel(const int4* __restrict__ cell, const unsigned* __restrict__ start,
                   unsigned* __restrict__ cursor, int* __restrict__ order, const int N) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const unsigned h = static_cast<unsigned>(cell[i].w);
    order[start[h] + atomicAdd(&cursor[h], 1u)] = i;
}

// Exclusive scan of n counters, two launches, blocks of kScanBlock elements (256 threads x 8):
// A writes every block's total; B sums the totals of the blocks before it (at most n / 2048
// values, read by all threads of the block) and scans its own elements on top of that.
constexpr int kScanBlock = 2048;

__device__ __forceinline__ unsigned lub_block_exclusive(unsigned v, unsigned* warp_sums, unsigned& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[w] = inc;
    __syncthreads();
    unsigned base = 0;
    total = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const unsigned ws = warp_sums[q];
        if (q < w) base += ws;
        total += ws;
    }
    __syncthreads();
    return base + inc - v;
}

__global__ void __launch_bounds__(256)
lub_scan_totals_kernel(const unsigned* __restrict__ count, unsigned* __restrict__ totals, const unsigned n) {
    __shared__ unsigned warp_sums[8];
    const unsigned b0 = blockIdx.x * kScanBlock + threadIdx.x * 8;
    unsigned v = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) v += (b0 + q < n) ? count[b0 + q] : 0u;
    unsigned total;
    lub_block_exclusive(v, warp_sums, total);
    if (threadIdx.x == 0) totals[blockIdx.x] = total;
}

__global__ void __launch_bounds__(256)
lub_scan_apply_kernel(const unsigned* __restrict__ count, const unsigned* __restrict__ totals,
                      unsigned* __restrict__ start, const unsigned n) {
    __shared__ unsigned warp_sums[8];
    __shared__ unsigned s_prefix;
    unsigned pre = 0;
    for (unsigned k = threadIdx.x; k < blockIdx.x; k += 256) pre += totals[k];
    unsigned dummy;
    const unsigned ex = lub_block_exclusive(pre, warp_sums, dummy);
    if (threadIdx.x == 255) s_prefix = ex + pre;
    __syncthreads();
    const unsigned prefix = s_prefix;
    const unsigned b0 = blockIdx.x * kScanBlock + threadIdx.x * 8;
    unsigned c[8], v = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        c[q] = (b0 + q < n) ? count[b0 + q] : 0u;
        v += c[q];
    }
    unsigned run = prefix + lub_block_exclusive(v, warp_sums, dummy);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (b0 + q < n) start[b0 + q] = run;
        run += c[q];
    }
}

// one thread per bucket: insertion sort by particle index (buckets hold a handful of particles)
__global__ void __launch_bounds__(256)
lub_sort_kernel(const unsigned* __restrict__ start, int* __restrict__ order, const unsigned H) {
    const unsigned h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= H) return;
    const unsigned b = start[h], e = start[h + 1];
    for (unsigned k = b + 1; k < e; ++k) {
        const int v = order[k];
        unsigned m = k;
        while (m > b && order[m - 1] > v) {
            order[m] = order[m - 1];
            --m;
        }
        order[m] = v;
    }
}

// sorted copies: particle data in bucket order, so that the force kernel reads contiguous runs
template <typename T4>
__global__ void __launch_bounds__(256)
lub_gather_kernel(const T4* __restrict__ pos, const T4* __restrict__ vel, const int4* __restrict__ cell,
                  const int* __restrict__ order, T4* __restrict__ spos, T4* __restrict__ svel,
                  int4* __restrict__ scell, const int N) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int i = order[k];
    spos[k] = pos[i];
    svel[k] = vel[i];
    int4 c = cell[i];
    c.w = i;  // the particle's own index travels with its cell
    scell[k] = c;
}

// nearest-image displacement of one component as a double, by the rule of the pair kernels
// (reading B2): fp32 modes decide n on the fp32 difference, fp64 on the double one.
template <typename S>
__device__ __forceinline__ double lub_disp(const S xi, const S xj, const LubGrid& g);
template <>
__device__ __forceinline__ double lub_disp<float>(const float xi, const float xj, const LubGrid& g) {
    if (g.nc == 0) return static_cast<double>(xi) - static_cast<double>(xj);
    const float d = __fsub_rn(xi, xj);
    const float Lf = static_cast<float>(g.L);
    const float n = __fsub_rn(__fmaf_rn(d, __fdiv_rn(1.0f, Lf), 12582912.0f), 12582912.0f);
    // only the image index n is an fp32 decision; the displacement is the exact difference of the
    // stored coordinates shifted by n box sides (all three terms are exact in double)
    return (static_cast<double>(xi) - static_cast<double>(xj)) - static_cast<double>(n) * static_cast<double>(Lf);
}
template <>
__device__ __forceinline__ double lub_disp<double>(const double xi, const double xj, const LubGrid& g) {
    const double d = xi - xj;
    if (g.nc == 0) return d;
    const double n = __dsub_rn(fma(d, g.invL, 6755399441055744.0), 6755399441055744.0);
    return __dsub_rn(d, __dmul_rn(n, g.L));
}

// r^2 < 9 a^2 decided in the arithmetic of the context (reading C3)
__device__ __forceinline__ bool lub_inside(float, double dx, double dy, double dz, double nine_a2) {
    const float fx = static_cast<float>(dx), fy = static_cast<float>(dy), fz = static_cast<float>(dz);
    return __fmaf_rn(fz, fz, __fmaf_rn(fy, fy, __fmul_rn(fx, fx))) < static_cast<float>(nine_a2);
}
__device__ __forceinline__ bool lub_inside(double, double dx, double dy, double dz, double nine_a2) {
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)) < nine_a2;
}

// fp32 contexts: a conservative pre-filter that never leaves fp32.  The decision itself is taken
// by lub_inside on the floats of the exact image displacement; the all-fp32 displacement used here
// differs from those by a few ulp of the box side, so candidates are only rejected when they lie
// outside 3a by a relative margin of 2^-10 in r^2 (>> ulp(L) / 3a for any box whose coordinates
// fp32 can still tell apart): ~95 % of the candidates go before any fp64 instruction is issued.
__device__ __forceinline__ bool lub_reject_f32(const float4 pi, const float4 pj, const LubGrid& g,
                                               const float nine_a2) {
    float dx = __fsub_rn(pi.x, pj.x), dy = __fsub_rn(pi.y, pj.y), dz = __fsub_rn(pi.z, pj.z);
    if (g.nc > 0) {
        const float Lf = static_cast<float>(g.L), iL = __fdiv_rn(1.0f, Lf), M = 12582912.0f;
        dx = __fmaf_rn(-__fsub_rn(__fmaf_rn(dx, iL, M), M), Lf, dx);
        dy = __fmaf_rn(-__fsub_rn(__fmaf_rn(dy, iL, M), M), Lf, dy);
        dz = __fmaf_rn(-__fsub_rn(__fmaf_rn(dz, iL, M), M), Lf, dz);
    }
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx))) > nine_a2 * 1.0009765625f;
}
__device__ __forceinline__ bool lub_reject_f32(const double4, const double4, const LubGrid&, const float) {
    return false;  // fp64 contexts decide in fp64 below
}

// force_out = F^ext - C.  fext: per-particle external forces or NULL (uniform g); fext may be
// force_out itself (each thread reads its own element before it writes it).
// LPP lanes per particle split the 27 neighbour cells (cell c goes to lane c mod LPP) and combine
// their sums by shuffles in a fixed order: with one lane per particle a small system leaves most
// SMs idle while every thread walks 27 cells and a dozen fp64 logarithms in sequence (84 us at
// N = 4000 on the fcc lattice, 12 neighbours inside 3a each).
template <typename T4, int LPP>
__global__ void __launch_bounds__(128, 8)
lub_force_kernel(const T4* __restrict__ spos, const T4* __restrict__ svel, const T4* fext,
                 const double gx, const double gy, const double gz, const int4* __restrict__ scell,
                 const unsigned* __restrict__ start, T4* force_out, const LubGrid g, const double a,
                 const double mu0, const int N) {
    typedef typename Vec4<T4>::S S;
    const int t0 = blockIdx.x * blockDim.x + threadIdx.x;
    const int sub = t0 % LPP;
    const bool live = t0 / LPP < N;
    const int k0 = live ? t0 / LPP : N - 1;  // idle lanes shadow the last particle, write nothing
    // thread k0 owns the k0-th particle in bucket order: the lanes of a warp sit in the same or in
    // neighbouring cells, probe the same buckets and read the same runs of the sorted copies
    const T4 pi = spos[k0];
    const T4 vi = svel[k0];
    const int4 ci = scell[k0];
    const int i = ci.w;
    const double nine_a2 = 9.0 * a * a, inv_a = 1.0 / a, inv_mu0 = 1.0 / mu0;
    double cx = 0.0, cy = 0.0, cz = 0.0;
    for (int c = sub; c < 27; c += LPP) {
                const int ox = c % 3 - 1, oy = (c / 3) % 3 - 1, oz = c / 9 - 1;
                int nx = ci.x + ox, ny = ci.y + oy, nz = ci.z + oz;
                if (g.nc > 0) {
                    nx = (nx + g.nc) % g.nc;
                    ny = (ny + g.nc) % g.nc;
                    nz = (nz + g.nc) % g.nc;
                }
                const unsigned h = lub_hash(nx, ny, nz, g.mask);
                const unsigned e = start[h + 1];
                for (unsigned k = start[h]; k < e; ++k) {
                    const int4 cj = scell[k];
                    if (cj.w == i || cj.x != nx || cj.y != ny || cj.z != nz) continue;  // self / alias
                    const T4 pj = spos[k];
                    if (sizeof(S) == 4 && lub_reject_f32(pi, pj, g, static_cast<float>(nine_a2))) continue;
                    const double dx = lub_disp<S>(pi.x, pj.x, g), dy = lub_disp<S>(pi.y, pj.y, g),
                                 dz = lub_disp<S>(pi.z, pj.z, g);
                    if (!lub_inside(S(0), dx, dy, dz, nine_a2)) continue;
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    if (r2 == 0.0) continue;  // coincident centres: no direction, no term
                    const double r = sqrt(r2);
                    double s = r * inv_a - 2.0;
                    s = s < kLubSmin ? kLubSmin : s;
                    const double ls = log(s);
                    const double par = (0.25 / s - 0.225 * ls) * inv_mu0;
                    const double per = (-ls * (1.0 / 6.0)) * inv_mu0;
                    const T4 vj = svel[k];
                    const double wx = static_cast<double>(vi.x) - static_cast<double>(vj.x);
                    const double wy = static_cast<double>(vi.y) - static_cast<double>(vj.y);
                    const double wz = static_cast<double>(vi.z) - static_cast<double>(vj.z);
                    const double rw = (dx * wx + dy * wy + dz * wz) / r2;
                    cx += per * wx + (par - per) * rw * dx;
                    cy += per * wy + (par - per) * rw * dy;
                    cz += per * wz + (par - per) * rw * dz;
                }
            }
#pragma unroll
    for (int o = LPP / 2; o > 0; o >>= 1) {
        cx += __shfl_xor_sync(0xffffffffu, cx, o, LPP);
        cy += __shfl_xor_sync(0xffffffffu, cy, o, LPP);
        cz += __shfl_xor_sync(0xffffffffu, cz, o, LPP);
    }
    if (!live || sub != 0) return;
    double fx = gx, fy = gy, fz = gz;
    if (fext) {
        const T4 f = fext[i];
        fx = f.x, fy = f.y, fz = f.z;
    }
    force_out[i] = Vec4<T4>::make(S(fx - cx), S(fy - cy), S(fz - cz), S(0));
}

// ---- small systems: all pairs in one launch ---------------------------------------------------
// Below a few thousand particles the seven launches of the cell grid cost more (~22 us even when
// replayed from a graph) than testing every pair: one warp per particle i, lane l takes
// j = l, l + 32, ...; same decision rule, same fp64 pair term, lane sums combined by shuffles in a
// fixed order.  N <= kLubSmallMax.
constexpr int kLubSmallMax = 2560;

template <typename T4>
__global__ void __launch_bounds__(256)
lub_small_kernel(const T4* __restrict__ pos, const T4* __restrict__ vel, const T4* fext,
                 const double gx, const double gy, const double gz, T4* force_out,
                 const LubGrid g, const double a, const double mu0, const int N) {
    typedef typename Vec4<T4>::S S;
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= N) return;  // whole warps leave together
    const T4 pi = pos[i];
    const T4 vi = vel[i];
    const double nine_a2 = 9.0 * a * a, inv_a = 1.0 / a, inv_mu0 = 1.0 / mu0;
    double cx = 0.0, cy = 0.0, cz = 0.0;
    for (int j = lane; j < N; j += 32) {
        if (j == i) continue;
        const T4 pj = pos[j];
        if (sizeof(S) == 4 && lub_reject_f32(pi, pj, g, static_cast<float>(nine_a2))) continue;
        const double dx = lub_disp<S>(pi.x, pj.x, g), dy = lub_disp<S>(pi.y, pj.y, g),
                     dz = lub_disp<S>(pi.z, pj.z, g);
        if (!lub_inside(S(0), dx, dy, dz, nine_a2)) continue;
        const double r2 = dx * dx + dy * dy + dz * dz;
        if (r2 == 0.0) continue;
        const double r = sqrt(r2);
        double s = r * inv_a - 2.0;
        s = s < kLubSmin ? kLubSmin : s;
        const double ls = log(s);
        const double par = (0.25 / s - 0.225 * ls) * inv_mu0;
        const double per = (-ls * (1.0 / 6.0)) * inv_mu0;
        const T4 vj = vel[j];
        const double wx = static_cast<double>(vi.x) - static_cast<double>(vj.x);
        const double wy = static_cast<double>(vi.y) - static_cast<double>(vj.y);
        const double wz = static_cast<double>(vi.z) - static_cast<double>(vj.z);
        const double rw = (dx * wx + dy * wy + dz * wz) / r2;
        cx += per * wx + (par - per) * rw * dx;
        cy += per * wy + (par - per) * rw * dy;
        cz += per * wz + (par - per) * rw * dz;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cx += __shfl_xor_sync(0xffffffffu, cx, o);
        cy += __shfl_xor_sync(0xffffffffu, cy, o);
        cz += __shfl_xor_sync(0xffffffffu, cz, o);
    }
    if (lane != 0) return;
    double fx = gx, fy = gy, fz = gz;
    if (fext) {
        const T4 f = fext[i];
        fx = f.x, fy = f.y, fz = f.z;
    }
    force_out[i] = Vec4<T4>::make(S(fx - cx), S(fy - cy), S(fz - cz), S(0));
}

}  // namespace sd
