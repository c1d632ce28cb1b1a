// sd_lub.cuh -- lubrication correction of the forces.
//
//   mu0 f_sing(r_ij) = [ 1/(4 s) - (9/40) ln s ] rr^ - (1/6) ln s (I - rr^) ,  s = r_ij / a - 2   Eq. (8)
//   F_i <- F_i^ext - sum'_j f_sing(r_ij) . (v_i - v_j)         step 2 of the paper's loop
//
// with the velocities of the previous product and the primed sum over j != i with r_ij < 3a
// ("we truncate ad hoc at s = 1 or r = 3a").  The paper points to Verlet lists and particle
// reordering for this O(N) step; here it is a cell grid rebuilt on every
// call, no host synchronisation, no memset, deterministic:
//   cells of side >= 3a; a cell (cx, cy, cz) goes to bucket  cx' + M (cy' + M cz'),  c' = c mod M,
//   M^3 = H = 8^k >= N buckets (periodic box: M = min(floor(L / 3a), 2^k) cells per edge, no
//   aliasing).  Buckets are x-major: the three x-neighbours of a cell are ONE contiguous run of
//   the sorted particle arrays, a particle probes 9 runs instead of 27 cells.  In free space cells
//   M apart share a bucket; their particles are >= (M - 2) cell sides >= 18 a away in that
//   coordinate and fail the distance test like any other candidate: no cell is stored anywhere.
//   lub_count_kernel    bucket of every particle (kept, 4 bytes each), bucket histogram by atomicAdd
//   lub_scan_*_kernel   exclusive scan of the H counters in two launches (block totals, then every
//                       block adds the totals before it to its own scan), written twice: bucket
//                       starts and the scatter cursors
//   lub_scatter_kernel  particle indices into their buckets (atomic cursor), then
//   lub_gather_kernel   positions and velocities copied into bucket order (the paper's
//                       "particle reordering": neighbouring cells are neighbouring memory), within
//                       a bucket by particle index (every thread ranks its particle among those
//                       of its bucket): the summation order below, and with it every bit of the
//                       result, does not depend on the atomics; clears the histogram for the
//                       next call
//   lub_force_kernel    particles in bucket order.  N large, one lane per particle: the lane walks
//                       its 9 runs with an all-fp32 test (fp64 contexts: the fp64 decision) and
//                       queues the candidates that pass in shared memory; the warp then evaluates
//                       the queued pairs of all its lanes 32 at a time, all lanes busy (Eq. 8 in
//                       fp64 with its logarithm costs ~300 instructions: evaluated where it was
//                       found, 1.35 hits per particle kept a warp in that divergent code for most
//                       of its life), and every lane adds its own terms in the order it found them.
//                       N small: 8 / 32 lanes per particle split the 27 cells and evaluate in place.
//                       The cut-off r^2 < 9a^2 is decided in the arithmetic of the context (fp32
//                       fma chain in the fp32 modes, reading C3) on the exact difference
//                       of the stored coordinates; sums in fp64 in a fixed order; writes F^ext - C
//                       rounded to the element type.
//   lub_one_launch_kernel   1024 < N <= 4096: all of the above in ONE launch, every CTA building the
//                       grid for itself in shared memory (see there)
//   lub_small_kernel    N <= 1024 (and boxes below 9a up to N = 4096): all pairs, one launch
// Periodic box: neighbour cells wrap, displacements take the nearest image by the rule of the
// pair kernels.  Measurements: profiles/r02_lubrication.md.
#pragma once
#include "sd_common.cuh"
#include "sd_stream.cuh"

namespace sd {

constexpr double kLubSmin = 1.0e-3;  // lower clamp of s (reading C2: Eq. 8 diverges at contact)

struct LubGrid {
    double inv_cell;  // 1 / cell side (free space)
    double L, invL;   // periodic cube (0: free space)
    int nc;           // cells per edge in the box (0: free space, unbounded integer cells)
    int M;            // bucket rows: cell coordinates enter the bucket index modulo M (box: M = nc)
};

// cell coordinate of x, already reduced modulo M (free space: M is a power of two)
__device__ __forceinline__ int lub_cell_coord(double x, const LubGrid& g) {
    if (g.nc > 0) {
        double u = x * g.invL;
        u -= floor(u);  // [0, 1)
        const int c = static_cast<int>(u * g.nc);
        return c < g.nc ? c : g.nc - 1;
    }
    return static_cast<int>(floor(x * g.inv_cell)) & (g.M - 1);
}
__device__ __forceinline__ unsigned lub_bucket(int cx, int cy, int cz, int M) {
    return static_cast<unsigned>(cx + M * (cy + M * cz));
}
__device__ __forceinline__ int lub_wrap(int c, int M) { return c < 0 ? c + M : (c >= M ? c - M : c); }

template <typename T4>
__device__ __forceinline__ unsigned lub_bucket_of(const T4 p, const LubGrid& g) {
    return lub_bucket(lub_cell_coord(p.x, g), lub_cell_coord(p.y, g), lub_cell_coord(p.z, g), g.M);
}

template <typename T4>
__global__ void __launch_bounds__(256)
lub_count_kernel(const T4* __restrict__ pos, unsigned* __restrict__ bucket, unsigned* __restrict__ count,
                 const LubGrid g, const int N) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const unsigned h = lub_bucket_of(pos[i], g);
    bucket[i] = h;
    atomicAdd(&count[h], 1u);
}

// cursor[h] starts at start[h] (lub_scan_apply_kernel).  slots[k] = (particle, bucket) of slot k:
// grouped by bucket, in the order the atomics happened to give within a bucket
__global__ void __launch_bounds__(256)
lub_scatter_kernel(const unsigned* __restrict__ bucket, unsigned* __restrict__ cursor,
                   int2* __restrict__ slots, const int N) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const unsigned h = bucket[i];
    slots[atomicAdd(&cursor[h], 1u)] = make_int2(i, static_cast<int>(h));
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

// eight consecutive counters of a thread as two 16-byte loads (the arrays come from cudaMalloc and
// b0 is a multiple of 8); the last, partial group of the array element by element
__device__ __forceinline__ void lub_load8(const unsigned* __restrict__ count, const unsigned b0, const unsigned n,
                                          unsigned (&c)[8]) {
    if (b0 + 8 <= n) {
        const uint4 lo = *reinterpret_cast<const uint4*>(count + b0);
        const uint4 hi = *reinterpret_cast<const uint4*>(count + b0 + 4);
        c[0] = lo.x, c[1] = lo.y, c[2] = lo.z, c[3] = lo.w, c[4] = hi.x, c[5] = hi.y, c[6] = hi.z, c[7] = hi.w;
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) c[q] = (b0 + q < n) ? count[b0 + q] : 0u;
    }
}

__global__ void __launch_bounds__(256)
lub_scan_totals_kernel(const unsigned* __restrict__ count, unsigned* __restrict__ totals, const unsigned n) {
    __shared__ unsigned warp_sums[8];
    const unsigned b0 = blockIdx.x * kScanBlock + threadIdx.x * 8;
    unsigned c[8], v = 0;
    lub_load8(count, b0, n, c);
#pragma unroll
    for (int q = 0; q < 8; ++q) v += c[q];
    unsigned total;
    lub_block_exclusive(v, warp_sums, total);
    if (threadIdx.x == 0) totals[blockIdx.x] = total;
}

// start[0 .. n) and cursor[0 .. n - 1): the same exclusive scan (n = H + 1: start[H] = N)
__global__ void __launch_bounds__(256)
lub_scan_apply_kernel(const unsigned* __restrict__ count, const unsigned* __restrict__ totals,
                      unsigned* __restrict__ start, unsigned* __restrict__ cursor, const unsigned n) {
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
    lub_load8(count, b0, n, c);
#pragma unroll
    for (int q = 0; q < 8; ++q) v += c[q];
    unsigned run = prefix + lub_block_exclusive(v, warp_sums, dummy);
    unsigned o[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        o[q] = run;
        run += c[q];
    }
    if (b0 + 8 < n) {  // all eight starts and all eight cursors exist
        const uint4 lo = make_uint4(o[0], o[1], o[2], o[3]), hi = make_uint4(o[4], o[5], o[6], o[7]);
        *reinterpret_cast<uint4*>(start + b0) = lo;
        *reinterpret_cast<uint4*>(start + b0 + 4) = hi;
        *reinterpret_cast<uint4*>(cursor + b0) = lo;
        *reinterpret_cast<uint4*>(cursor + b0 + 4) = hi;
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            if (b0 + q < n) start[b0 + q] = o[q];
            if (b0 + q + 1 < n) cursor[b0 + q] = o[q];
        }
    }
}

// insertion sort of order[b, e) by particle index (buckets hold a handful of particles)
__device__ __forceinline__ void lub_sort_run(int* order, const unsigned b, const unsigned e) {
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

// Sorted copies: particle data in bucket order, so that the force kernel reads contiguous runs,
// and within a bucket in the order of the particle index: the summation order of the force
// kernel, and with it every bit of the result, does not depend on the atomics of the scatter.
// Thread k takes the particle the scatter left in slot k, finds its rank among the (handful of)
// particles of its bucket and writes it to slot start + rank; the first slot of every bucket also
// clears the bucket's counter for the next call.
template <typename T4>
__global__ void __launch_bounds__(256)
lub_gather_kernel(const T4* __restrict__ pos, const T4* __restrict__ vel, const int2* __restrict__ slots,
                  const unsigned* __restrict__ start, unsigned* __restrict__ count, int* __restrict__ order,
                  T4* __restrict__ spos, T4* __restrict__ svel, const int N) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int2 me = slots[k];
    const T4 p = pos[me.x];
    const T4 v = vel[me.x];
    const unsigned b = start[me.y], e = start[me.y + 1];
    if (static_cast<unsigned>(k) == b) count[me.y] = 0u;
    unsigned slot = b;
    for (unsigned q = b; q < e; ++q) slot += slots[q].x < me.x ? 1u : 0u;
    order[slot] = me.x;
    spos[slot] = p;
    svel[slot] = v;
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
// The loop-invariant floats of the test are set up once by the caller:
struct LubCut {
    float cut;      // 9 a^2 (1 + 2^-10)
    float Lf, iLf;  // box side and its reciprocal (box only)
    bool box;
};
__device__ __forceinline__ LubCut lub_cut_f32(const double nine_a2, const LubGrid& g) {
    LubCut c;
    c.cut = static_cast<float>(nine_a2) * 1.0009765625f;
    c.box = g.nc > 0;
    c.Lf = static_cast<float>(g.L);
    c.iLf = c.box ? __fdiv_rn(1.0f, c.Lf) : 0.0f;
    return c;
}
__device__ __forceinline__ bool lub_reject_f32(const float4 pi, const float4 pj, const LubCut& c) {
    float dx = __fsub_rn(pi.x, pj.x), dy = __fsub_rn(pi.y, pj.y), dz = __fsub_rn(pi.z, pj.z);
    if (c.box) {
        const float M = 12582912.0f;
        dx = __fmaf_rn(-__fsub_rn(__fmaf_rn(dx, c.iLf, M), M), c.Lf, dx);
        dy = __fmaf_rn(-__fsub_rn(__fmaf_rn(dy, c.iLf, M), M), c.Lf, dy);
        dz = __fmaf_rn(-__fsub_rn(__fmaf_rn(dz, c.iLf, M), M), c.Lf, dz);
    }
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx))) > c.cut;
}
__device__ __forceinline__ bool lub_reject_f32(const double4, const double4, const LubCut&) {
    return false;  // fp64 contexts decide in fp64
}

// One pair's term of the sum: t = f_sing(r_ij) . (v_i - v_j), or zero if the pair is outside the
// cut-off (decided here, on the exact image displacement, in the arithmetic of the context) or the
// centres coincide (no direction, no term).
template <typename T4>
__device__ __forceinline__ void lub_pair_term(const T4 pi, const T4 vi, const T4 pj, const T4 vj,
                                              const LubGrid& g, const double nine_a2, const double inv_a,
                                              const double inv_mu0, double& tx, double& ty, double& tz) {
    typedef typename Vec4<T4>::S S;
    tx = ty = tz = 0.0;
    const double dx = lub_disp<S>(pi.x, pj.x, g), dy = lub_disp<S>(pi.y, pj.y, g),
                 dz = lub_disp<S>(pi.z, pj.z, g);
    if (!lub_inside(S(0), dx, dy, dz, nine_a2)) return;
    const double r2 = dx * dx + dy * dy + dz * dz;
    if (r2 == 0.0) return;
    const double r = sqrt(r2);
    double s = r * inv_a - 2.0;
    s = s < kLubSmin ? kLubSmin : s;
    const double ls = log(s);
    const double par = (0.25 / s - 0.225 * ls) * inv_mu0;
    const double per = (-ls * (1.0 / 6.0)) * inv_mu0;
    const double wx = static_cast<double>(vi.x) - static_cast<double>(vj.x);
    const double wy = static_cast<double>(vi.y) - static_cast<double>(vj.y);
    const double wz = static_cast<double>(vi.z) - static_cast<double>(vj.z);
    const double rw = (dx * wx + dy * wy + dz * wz) / r2;
    tx = per * wx + (par - per) * rw * dx;
    ty = per * wy + (par - per) * rw * dy;
    tz = per * wz + (par - per) * rw * dz;
}

// cheap test of a candidate before it is queued: fp32 contexts the all-fp32 pre-filter, fp64
// contexts the decision itself
__device__ __forceinline__ bool lub_candidate(const float4 pi, const float4 pj, const LubGrid&,
                                              const LubCut& c, const double) {
    return !lub_reject_f32(pi, pj, c);
}
__device__ __forceinline__ bool lub_candidate(const double4 pi, const double4 pj, const LubGrid& g,
                                              const LubCut&, const double nine_a2) {
    return lub_inside(0.0, lub_disp<double>(pi.x, pj.x, g), lub_disp<double>(pi.y, pj.y, g),
                      lub_disp<double>(pi.z, pj.z, g), nine_a2);
}

constexpr int kLubThreads = 128;        // lub_force_kernel
constexpr int kLubQ = 8;                // queued candidates per lane between two evaluation rounds
constexpr int kLubOneLaneMinN = 49152;  // one lane per particle (queued evaluation) from here on

__device__ __forceinline__ void lub_prefetch(const void* p) {
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
}

struct LubWarpQueue {
    int k[kLubQ][32];    // queued candidates, [slot][lane]
    double t[3][32];     // terms of one evaluation round
    unsigned pre[32];    // first round slot of every lane
};

// All 32 lanes of a warp: evaluate the queued pairs of the warp, 32 per round, every lane busy;
// returns the sum of the calling lane's own terms, added in the order they were queued.
template <typename T4>
__device__ __forceinline__ double3 lub_flush(LubWarpQueue* q, const T4* __restrict__ spos,
                                             const T4* __restrict__ svel, const int nq, const int kw0,
                                             const LubGrid& g, const double nine_a2, const double inv_a,
                                             const double inv_mu0) {
    const int lane = threadIdx.x & 31;
    unsigned incl = static_cast<unsigned>(nq);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    const unsigned excl = incl - static_cast<unsigned>(nq);
    const unsigned total = __shfl_sync(0xffffffffu, incl, 31);
    q->pre[lane] = excl;
    __syncwarp();
    double3 acc = make_double3(0.0, 0.0, 0.0);
    for (unsigned base = 0; base < total; base += 32) {
        const unsigned t = base + lane;
        double tx = 0.0, ty = 0.0, tz = 0.0;
        if (t < total) {
            int owner = 0;  // the last lane whose first slot is <= t (it has a non-empty queue)
#pragma unroll
            for (int step = 16; step > 0; step >>= 1)
                if (q->pre[owner + step] <= t) owner += step;
            const int kj = q->k[t - q->pre[owner]][owner];
            const int ko = kw0 + owner;
            lub_pair_term(spos[ko], svel[ko], spos[kj], svel[kj], g, nine_a2, inv_a, inv_mu0, tx, ty, tz);
        }
        q->t[0][lane] = tx, q->t[1][lane] = ty, q->t[2][lane] = tz;
        __syncwarp();
        const unsigned lo = max(excl, base), hi = min(excl + static_cast<unsigned>(nq), base + 32u);
        for (unsigned u = lo; u < hi; ++u)
            acc.x += q->t[0][u - base], acc.y += q->t[1][u - base], acc.z += q->t[2][u - base];
        __syncwarp();
    }
    return acc;
}

// force_out = F^ext - C.  fext: per-particle external forces or NULL (uniform g); fext may be
// force_out itself (each thread reads its own element before it writes it).
// LPP lanes per particle.  LPP = 1: see the header.  LPP = 8 / 32: the lanes split the 27 neighbour
// cells (cell c goes to lane c mod LPP), evaluate in place and combine their sums by shuffles in a
// fixed order: with one lane per particle a small system leaves most SMs idle.
template <typename T4, int LPP>
__global__ void __launch_bounds__(kLubThreads, 8)
lub_force_kernel(const T4* __restrict__ spos, const T4* __restrict__ svel, const int* __restrict__ order,
                 const T4* fext, const double gx, const double gy, const double gz,
                 const unsigned* __restrict__ start, T4* force_out, const LubGrid g, const double a,
                 const double mu0, const int N) {
    typedef typename Vec4<T4>::S S;
    __shared__ LubWarpQueue queues[LPP == 1 ? kLubThreads / 32 : 1];
    const int t0 = blockIdx.x * blockDim.x + threadIdx.x;
    const int sub = t0 % LPP;
    const bool live = t0 / LPP < N;
    const int k0 = live ? t0 / LPP : N - 1;  // idle lanes shadow the last particle, write nothing
    // thread k0 owns the k0-th particle in bucket order: the lanes of a warp sit in the same or in
    // neighbouring cells and read the same runs of the sorted copies
    const T4 pi = spos[k0];
    const T4 vi = svel[k0];
    const int M = g.M;
    const int cxm = lub_cell_coord(pi.x, g), cym = lub_cell_coord(pi.y, g), czm = lub_cell_coord(pi.z, g);
    const double nine_a2 = 9.0 * a * a, inv_a = 1.0 / a, inv_mu0 = 1.0 / mu0;
    const LubCut cut = lub_cut_f32(nine_a2, g);
    double cx = 0.0, cy = 0.0, cz = 0.0;
    if (LPP == 1) {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int kw0 = t0 - lane;  // sorted index of lane 0's particle
        int nq = 0;
        LubWarpQueue* q = &queues[warp];
        int* qpush = &q->k[0][lane];  // slot s of this lane: qpush[32 s]
        auto flush = [&]() {
            const double3 t = lub_flush<T4>(q, spos, svel, nq, kw0, g, nine_a2, inv_a, inv_mu0);
            cx += t.x, cy += t.y, cz += t.z;
            nq = 0;
        };
        // the lane's runs of candidates: 9 rows of three x-neighbours (a row that wraps in x is two
        // runs), their 18 - 36 bucket bounds fetched in one go, empty runs dropped
        unsigned rb[18], re[18];
        int nr = 0;
        if (live) {
            const int xa = cxm - 1, xb = cxm + 1;
            const int a0 = max(xa, 0), a1 = min(xb, M - 1) + 1;
            const int xw = xa < 0 ? M - 1 : (xb >= M ? 0 : -1);  // the cell across the end of the row
            unsigned b[9], e[9];
#pragma unroll
            for (int r = 0; r < 9; ++r) {
                const int ny = lub_wrap(cym + r % 3 - 1, M), nz = lub_wrap(czm + r / 3 - 1, M);
                const unsigned row = static_cast<unsigned>(M * (ny + M * nz));
                b[r] = start[row + a0], e[r] = start[row + a1];
            }
#pragma unroll
            for (int r = 0; r < 9; ++r)
                if (b[r] < e[r]) {
                    rb[nr] = b[r], re[nr] = e[r], ++nr;
                    lub_prefetch(spos + b[r]);  // the head of every run is on its way before the loop starts
                }
            if (xw >= 0) {
#pragma unroll
                for (int r = 0; r < 9; ++r) {
                    const int ny = lub_wrap(cym + r % 3 - 1, M), nz = lub_wrap(czm + r / 3 - 1, M);
                    const unsigned row = static_cast<unsigned>(M * (ny + M * nz));
                    b[r] = start[row + xw], e[r] = start[row + xw + 1];
                }
#pragma unroll
                for (int r = 0; r < 9; ++r)
                    if (b[r] < e[r]) rb[nr] = b[r], re[nr] = e[r], ++nr;
            }
        }
        // one candidate per lane and iteration, the next one and the bounds of the next run already
        // on their way; the loop is warp-uniform, so the warp can stop and evaluate as soon as one
        // lane's queue is full
        unsigned k = 0, e = 0, nb = 0, ne = 0;
        int r = 2;
        if (nr > 0) k = rb[0], e = re[0];
        if (nr > 1) nb = rb[1], ne = re[1];
        bool have = k < e;
        T4 pj = have ? spos[k] : pi;
#pragma unroll 1
        while (__any_sync(0xffffffffu, have)) {
            if (__any_sync(0xffffffffu, nq == kLubQ)) flush();
            const unsigned kc = k;
            const T4 pc = pj;
            const bool hc = have;
            {  // advance, branch-free: runs are short, some lane switches runs in almost every iteration
                k += have ? 1u : 0u;
                const bool sw = have && k >= e;
                const int rr = r < 17 ? r : 17;
                const unsigned tb = rb[rr], te = re[rr];
                const bool more = r < nr;
                k = sw ? nb : k, e = sw ? ne : e;
                nb = sw ? (more ? tb : 0u) : nb, ne = sw ? (more ? te : 0u) : ne;
                r += sw ? 1 : 0;
                have = k < e;
                if (have) pj = spos[k];
            }
            if (hc && static_cast<int>(kc) != k0 && lub_candidate(pi, pc, g, cut, nine_a2)) {
                qpush[32 * nq] = static_cast<int>(kc);
                ++nq;
            }
        }
        if (__any_sync(0xffffffffu, nq > 0)) flush();
    } else {
        for (int c = sub; c < 27; c += LPP) {
            const int nx = lub_wrap(cxm + c % 3 - 1, M), ny = lub_wrap(cym + (c / 3) % 3 - 1, M),
                      nz = lub_wrap(czm + c / 9 - 1, M);
            const unsigned h = lub_bucket(nx, ny, nz, M);
            const unsigned e = start[h + 1];
            for (unsigned k = start[h]; k < e; ++k) {
                if (static_cast<int>(k) == k0) continue;
                const T4 pj = spos[k];
                const T4 vj = svel[k];  // with the position, not after the test: one round trip less
                if (sizeof(S) == 4 && !lub_candidate(pi, pj, g, cut, nine_a2)) continue;
                double tx, ty, tz;
                lub_pair_term(pi, vi, pj, vj, g, nine_a2, inv_a, inv_mu0, tx, ty, tz);
                cx += tx, cy += ty, cz += tz;
            }
        }
#pragma unroll
        for (int o = LPP / 2; o > 0; o >>= 1) {
            cx += __shfl_xor_sync(0xffffffffu, cx, o, LPP);
            cy += __shfl_xor_sync(0xffffffffu, cy, o, LPP);
            cz += __shfl_xor_sync(0xffffffffu, cz, o, LPP);
        }
    }
    if (!live || sub != 0) return;
    const int i = order[k0];
    double fx = gx, fy = gy, fz = gz;
    if (fext) {
        const T4 f = fext[i];
        fx = f.x, fy = f.y, fz = f.z;
    }
    force_out[i] = Vec4<T4>::make(S(fx - cx), S(fy - cy), S(fz - cz), S(0));
}

// ---- 1024 < N <= 4096: the whole step in ONE launch --------------------------------------------
// Every CTA builds the SAME cell grid for itself in shared memory (histogram, scan, scatter, sort by
// index, positions in bucket order: the five build kernels above in one CTA of 1024 threads, four
// particles per thread, phases separated by __syncthreads(); the 64 KB of positions come out of L2
// for all but the first CTA) and then takes its share of the particles, one warp per particle,
// the 27 neighbour cells on 27 lanes, candidates from shared memory.  A second launch and the
// round trip of the sorted copies through global memory cost more than 147 redundant builds that
// run side by side (profiles/r02_lubrication.md).
constexpr int kLubOneCtaThreads = 1024;
constexpr int kLubOneCtaPer = 4;  // particles per thread
constexpr int kLubOneCtaMaxN = kLubOneCtaThreads * kLubOneCtaPer;
constexpr unsigned kLubOneCtaMaxH = 4096;  // 16^3 buckets

template <typename T4>
struct LubOneLaunchSmem {
    unsigned cnt[kLubOneCtaMaxH];  // histogram, cursors, finally the end of every bucket
    int ord[kLubOneCtaMaxN];       // particle index of sorted slot k
    int inv[kLubOneCtaMaxN];       // sorted slot of particle i
    T4 sp[kLubOneCtaMaxN];         // positions in bucket order
    unsigned warp_sums[32];
};

template <typename T4>
__global__ void __launch_bounds__(kLubOneCtaThreads, 1)
lub_one_launch_kernel(const T4* __restrict__ pos, const T4* __restrict__ vel, const T4* fext, const double gx,
                      const double gy, const double gz, T4* force_out, const LubGrid g, const double a,
                      const double mu0, const int N) {
    typedef typename Vec4<T4>::S S;
    extern __shared__ __align__(16) unsigned char lub_smem_raw[];
    LubOneLaunchSmem<T4>& sm = *reinterpret_cast<LubOneLaunchSmem<T4>*>(lub_smem_raw);
    constexpr unsigned H = kLubOneCtaMaxH;
    const int tid = threadIdx.x;
    const int lane = tid & 31, w = tid >> 5;
    T4 p[kLubOneCtaPer];
#pragma unroll
    for (int q = 0; q < kLubOneCtaPer; ++q) {
        const int i = tid + kLubOneCtaThreads * q;
        if (i < N) p[q] = pos[i];
    }
#pragma unroll
    for (int q = 0; q < static_cast<int>(H) / kLubOneCtaThreads; ++q) sm.cnt[tid + kLubOneCtaThreads * q] = 0u;
    __syncthreads();
    unsigned hq[kLubOneCtaPer];
#pragma unroll
    for (int q = 0; q < kLubOneCtaPer; ++q) {
        if (tid + kLubOneCtaThreads * q < N) {
            hq[q] = lub_bucket_of(p[q], g);
            atomicAdd(&sm.cnt[hq[q]], 1u);
        }
    }
    __syncthreads();
    // exclusive scan: a thread owns `per` consecutive counters
    constexpr unsigned per = H / kLubOneCtaThreads;
    const unsigned b0 = tid * per;
    unsigned v = 0;
#pragma unroll
    for (unsigned q = 0; q < per; ++q) v += sm.cnt[b0 + q];
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) sm.warp_sums[w] = inc;
    __syncthreads();
    if (w == 0) {
        unsigned s = sm.warp_sums[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += t;
        }
        sm.warp_sums[lane] = s;  // inclusive
    }
    __syncthreads();
    unsigned run = (w ? sm.warp_sums[w - 1] : 0u) + inc - v;
#pragma unroll
    for (unsigned q = 0; q < per; ++q) {
        const unsigned c = sm.cnt[b0 + q];
        sm.cnt[b0 + q] = run;
        run += c;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kLubOneCtaPer; ++q) {
        const int i = tid + kLubOneCtaThreads * q;
        if (i < N) sm.ord[atomicAdd(&sm.cnt[hq[q]], 1u)] = i;
    }
    __syncthreads();
    // after the scatter cnt[h] is the END of bucket h, i.e. the start of bucket h + 1
#pragma unroll
    for (unsigned q = 0; q < per; ++q) {
        const unsigned h = tid + kLubOneCtaThreads * q;
        lub_sort_run(sm.ord, h ? sm.cnt[h - 1] : 0u, sm.cnt[h]);
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kLubOneCtaPer; ++q) {
        const int k = tid + kLubOneCtaThreads * q;
        if (k < N) sm.inv[sm.ord[k]] = k;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kLubOneCtaPer; ++q) {
        const int i = tid + kLubOneCtaThreads * q;
        if (i < N) sm.sp[sm.inv[i]] = p[q];
    }
    __syncthreads();

    // this CTA's particles (in bucket order), one warp each
    const int share = (N + gridDim.x - 1) / gridDim.x;
    const int k_end = min(N, static_cast<int>(blockIdx.x + 1) * share);
    const int M = g.M;
    const double nine_a2 = 9.0 * a * a, inv_a = 1.0 / a, inv_mu0 = 1.0 / mu0;
    const LubCut cut = lub_cut_f32(nine_a2, g);
    for (int k0 = blockIdx.x * share + w; k0 < k_end; k0 += kLubOneCtaThreads / 32) {
        const int i = sm.ord[k0];
        const T4 pi = sm.sp[k0];
        const T4 vi = vel[i];
        double cx = 0.0, cy = 0.0, cz = 0.0;
        if (lane < 27) {
            const int nx = lub_wrap(lub_cell_coord(pi.x, g) + lane % 3 - 1, M),
                      ny = lub_wrap(lub_cell_coord(pi.y, g) + (lane / 3) % 3 - 1, M),
                      nz = lub_wrap(lub_cell_coord(pi.z, g) + lane / 9 - 1, M);
            const unsigned h = lub_bucket(nx, ny, nz, M);
            const unsigned e = sm.cnt[h];
            for (unsigned k = h ? sm.cnt[h - 1] : 0u; k < e; ++k) {
                if (static_cast<int>(k) == k0) continue;
                const T4 pj = sm.sp[k];
                if (sizeof(S) == 4 && !lub_candidate(pi, pj, g, cut, nine_a2)) continue;
                double tx, ty, tz;
                lub_pair_term(pi, vi, pj, vel[sm.ord[k]], g, nine_a2, inv_a, inv_mu0, tx, ty, tz);
                cx += tx, cy += ty, cz += tz;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            cx += __shfl_xor_sync(0xffffffffu, cx, o);
            cy += __shfl_xor_sync(0xffffffffu, cy, o);
            cz += __shfl_xor_sync(0xffffffffu, cz, o);
        }
        if (lane == 0) {
            double fx = gx, fy = gy, fz = gz;
            if (fext) {
                const T4 f = fext[i];
                fx = f.x, fy = f.y, fz = f.z;
            }
            force_out[i] = Vec4<T4>::make(S(fx - cx), S(fy - cy), S(fz - cz), S(0));
        }
    }
}

// ---- small systems: all pairs in one launch ---------------------------------------------------
// Up to a thousand particles testing every pair costs less than building any grid: one warp per
// particle i, lane l takes j = l, l + 32, ...; same decision rule, same fp64 pair term, lane sums
// combined by shuffles in a fixed order.  N <= kLubSmallMax (measured on the fcc benchmark of the
// paper, full loop per step: N = 108 6.0 us against 10.9 with lub_one_launch_kernel, N = 864 17.1
// against 17.3, N = 2048 33.1 against 23.8); also boxes between 6a and 9a up to N = 4096.
constexpr int kLubSmallMax = 1024;

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
    const LubCut cut = lub_cut_f32(nine_a2, g);
    double cx = 0.0, cy = 0.0, cz = 0.0;
    for (int j = lane; j < N; j += 32) {
        if (j == i) continue;
        const T4 pj = pos[j];
        if (sizeof(S) == 4 && lub_reject_f32(pi, pj, cut)) continue;
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
