// sd_b200.cu -- C ABI (include/sd_b200.h), context, static schedule and kernel dispatcher.
//
// Host side only: every step of the hot path (pack, pair sums, reduction + self term,
// integrator update) runs in the kernels of sd_pairs_f32.cuh / sd_pairs_f64.cuh /
// sd_stream.cuh.  There is no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "../../include/sd_b200.h"
#include "sd_common.cuh"
#include "sd_pairs_f32.cuh"
#include "sd_pairs_f64.cuh"
#include "sd_pairs_f32w.cuh"
#include "sd_pairs_f64w.cuh"
#include "sd_access.cuh"
#include "sd_lub.cuh"
#include "sd_small.cuh"
#include "sd_stream.cuh"

namespace {

thread_local std::string g_create_error;

struct Config {
    int ipt = 0;        // particles i per thread
    int IB = 0;         // particles per i-block
    int TJ = 0;         // j per tile
    int B = 0, T = 0, G = 0;
    long long U = 0;
    int max_slots = 0;
    const void* kernel = nullptr;
    const char* name = "";
};

}  // namespace

namespace {
constexpr long long kGraphSteps = 16;  // even: the small-N Euler path ping-pongs two buffers
constexpr long long kGraphMaxN = 32768; // below: the gaps between launches are a measurable share of a step
struct GraphKey {  // everything a captured step sequence has baked in (besides the context state)
    void* pos;
    const void* force;
    double gx, gy, gz;
    bool has_gravity;
    double dt;
    int integrator;
};
}  // namespace

struct sd_ctx {
    long long N = 0;
    long long Nrec = 0;
    double a = 0, eta = 0, mu0 = 0;
    int tensor = SD_TENSOR_RPY;
    int precision = SD_PREC_F32_KAHAN;
    double box = 0.0;  // side of the periodic cube; 0 = free space
    long long small_apply_max = sd::kSmallApplyMax;  // N up to which the one-launch warp-per-particle kernel runs
    long long small_user = -1;                       // sd_set_dispatch override (< 0: automatic, see configure)
    int ipt_override = 0;                            // particles per thread; 0 = automatic
    int staging = 0;                                 // sd::STAGE_* (ablation, fp32 RPY Kahan only)
    int pos_comp = 1;                                // 0: plain fp32 positions (ablation)
    int lubrication = 0;                             // sd_step corrects the forces by Eq. (8)
    // lubrication cell grid (allocated on first use)
    unsigned* lub_bucket = nullptr;  // [N] bucket of every particle
    unsigned* lub_count = nullptr;   // [H + 1] bucket histogram (left zeroed by every call)
    unsigned* lub_start = nullptr;   // [H + 1] exclusive scan of it
    unsigned* lub_cursor = nullptr;  // [H]
    int2* lub_slots = nullptr;       // [N] (particle, bucket) grouped by bucket, as the scatter left them
    int* lub_order = nullptr;        // [N] particle indices grouped by bucket, sorted within a bucket
    void* lub_spos = nullptr;        // [N] positions, velocities in bucket order
    void* lub_svel = nullptr;
    bool lub_one_launch_ready = false;  // shared-memory attribute of lub_one_launch_kernel set
    bool lub_count_dirty = false;    // a call was abandoned between lub_count_kernel and lub_gather_kernel
    void* lub_tmp = nullptr;         // block totals of the bucket scan
    size_t lub_tmp_bytes = 0;
    unsigned lub_H = 0;
    // CUDA graph of kGraphSteps steps of the full loop (constant forces + lubrication)
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t gexec = nullptr;
    GraphKey gkey{};
    long long graph_launches = 0;
    int device = 0;
    int num_sms = 0;
    Config cfg;
    // warp-split one-launch kernel (sd_pairs_f32w.cuh): its own schedule and scratch
    int jsplit = 0;             // 0 automatic, 1 classic tiled kernels only, 2 warp-split wherever it exists
    bool w_on = false;          // the current settings run through the warp-split kernel
    Config wcfg;
    size_t w_smem = 0;
    void* w_part = nullptr;
    int* w_blk_done = nullptr;
    long long* w_cta_u0 = nullptr;
    int* w_blk_first = nullptr;
    int* w_blk_nslots = nullptr;
    int* w_cta_piece = nullptr;
    void* w_pad = nullptr;      // 2 x kWSJ pad records: far-away positions | zero forces
    void* grav_buf = nullptr;   // uniform force written out per particle (sd_step with gravity)
    bool valid = false;         // false after a failed (re)configuration: every entry point refuses
    // device buffers (context-owned)
    void* rec = nullptr;        // packed records
    void* part = nullptr;       // segment partial sums
    void* vel = nullptr;        // velocities of the last product
    size_t vel_bytes = 0;
    void* pos_lo = nullptr;     // low words of the positions (fp32 modes)
    void* pos_half = nullptr;   // midpoint positions (for force callbacks)
    void* pos_alt = nullptr;    // ping-pong partner of pos (small-N Euler)
    void* force_buf = nullptr;  // forces written by a callback
    void* stage_pos = nullptr;  // device staging of the _host entry point
    void* stage_force = nullptr;
    void* stage_vel = nullptr;
    void* probe = nullptr;
    long long* d_cta_u0 = nullptr;
    int* d_blk_first = nullptr;
    int* d_blk_nslots = nullptr;
    int* d_cta_piece = nullptr;
    bool lo_valid = false;
    long long launches = 0;
    bool profiling = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_events;  // recorded, not yet read
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_pool;    // reusable
    std::string err;
};

namespace {

size_t elem_size(int precision) { return precision == SD_PREC_F64 ? sizeof(double) : sizeof(float); }

sd_status fail(sd_ctx* ctx, sd_status code, const std::string& msg) {
    if (ctx) ctx->err = msg;
    else g_create_error = msg;
    return code;
}

#define SD_CUDA(ctx, call)                                                                 \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess)                                                             \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? SD_ERR_ALLOC : SD_ERR_CUDA, \
                        std::string(#call) + ": " + cudaGetErrorString(e_));               \
    } while (0)

// Every entry point that touches the device: the context must be usable and the caller's current
// device must be the one the context was created on (its buffers and streams live there).
sd_status enter(sd_ctx* c, const char* who) {
    if (!c->valid)
        return fail(c, SD_ERR_INVALID_ARG, std::string(who) + ": the context is unusable after a failed "
                    "reconfiguration (" + c->err + "); call a setter that succeeds, or destroy it");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device)
        return fail(c, SD_ERR_INVALID_ARG, std::string(who) + ": the current CUDA device is not the one the "
                    "context was created on (cudaSetDevice first)");
    return SD_OK;
}
#define SD_ENTER(ctx, who)                      \
    do {                                        \
        sd_status e_ = enter(ctx, who);         \
        if (e_ != SD_OK) return e_;             \
    } while (0)

template <int I2, int TENSOR, int ACC, bool PBC, int TJ = sd::kTJ, int REPAIR = 1>
const void* f32_kernel() {
    return reinterpret_cast<const void*>(&sd::pairs_f32_kernel<I2, TENSOR, ACC, PBC, sd::STAGE_BULK, TJ, REPAIR>);
}
// 8 particles per thread at N >= kRepairMaxN: the round-1 careful pass (see sd_pairs_f32.cuh)
template <bool PBC>
const void* f32_pick_large(bool rpy, bool plain) {
    return rpy ? (plain ? f32_kernel<4, 0, 1, PBC, sd::kTJLarge, 0>() : f32_kernel<4, 0, 0, PBC, sd::kTJLarge, 0>())
               : (plain ? f32_kernel<4, 1, 1, PBC, sd::kTJLarge, 0>() : f32_kernel<4, 1, 0, PBC, sd::kTJLarge, 0>());
}
template <int I, int TENSOR, bool PBC, int TJ = sd::kTJ64>
const void* f64_kernel() {
    return reinterpret_cast<const void*>(&sd::pairs_f64_kernel<I, TENSOR, PBC, TJ>);
}
template <int I2, bool PBC, int TJ = sd::kTJ>
const void* f32_pick(bool rpy, bool plain) {
    return rpy ? (plain ? f32_kernel<I2, 0, 1, PBC, TJ>() : f32_kernel<I2, 0, 0, PBC, TJ>())
               : (plain ? f32_kernel<I2, 1, 1, PBC, TJ>() : f32_kernel<I2, 1, 0, PBC, TJ>());
}
template <int I, bool PBC, int TJ = sd::kTJ64>
const void* f64_pick(bool rpy) {
    return rpy ? f64_kernel<I, 0, PBC, TJ>() : f64_kernel<I, 1, PBC, TJ>();
}

void drop_graph(sd_ctx* c) {
    if (c->gexec) cudaGraphExecDestroy(c->gexec);
    c->gexec = nullptr;
}

void free_buffers(sd_ctx* c) {
    drop_graph(c);
    void** bufs[] = {&c->rec,       &c->part,        &c->vel,       &c->pos_lo, &c->pos_half, &c->pos_alt,
                     &c->force_buf, &c->stage_pos,   &c->stage_force, &c->stage_vel, &c->probe};
    for (void** b : bufs) {
        if (*b) cudaFree(*b);
        *b = nullptr;
    }
    void** lub[] = {reinterpret_cast<void**>(&c->lub_bucket), reinterpret_cast<void**>(&c->lub_count),
                    reinterpret_cast<void**>(&c->lub_start), reinterpret_cast<void**>(&c->lub_cursor),
                    reinterpret_cast<void**>(&c->lub_order), reinterpret_cast<void**>(&c->lub_slots), &c->lub_tmp,
                    &c->lub_spos, &c->lub_svel};
    for (void** b : lub) {
        if (*b) cudaFree(*b);
        *b = nullptr;
    }
    c->lub_H = 0;
    void** wb[] = {&c->w_part, reinterpret_cast<void**>(&c->w_blk_done), reinterpret_cast<void**>(&c->w_cta_u0),
                   reinterpret_cast<void**>(&c->w_blk_first), reinterpret_cast<void**>(&c->w_blk_nslots),
                   reinterpret_cast<void**>(&c->w_cta_piece), &c->w_pad, &c->grav_buf};
    for (void** b : wb) {
        if (*b) cudaFree(*b);
        *b = nullptr;
    }
    c->w_on = false;
    if (c->d_cta_u0) cudaFree(c->d_cta_u0);
    if (c->d_blk_first) cudaFree(c->d_blk_first);
    if (c->d_blk_nslots) cudaFree(c->d_blk_nslots);
    if (c->d_cta_piece) cudaFree(c->d_cta_piece);
    c->d_cta_piece = nullptr;
    c->d_cta_u0 = nullptr;
    c->d_blk_first = c->d_blk_nslots = nullptr;
}

// Static schedule of the tiled kernels (pure host code; also exported as sd_schedule_plan so that
// it can be tested without a GPU).  Units u = b * T + t over B i-blocks x T j-tiles; piece g of G
// owns units [u0[g], u0[g+1]); block b collects the partial sums of pieces first[b] ...
// first[b] + nslots[b] - 1; CTA blockIdx.x works on piece piece[blockIdx.x].
struct HostSchedule {
    int B = 0, T = 0, G = 0, max_slots = 1;
    long long U = 0;
    std::vector<long long> u0;
    std::vector<int> first, nslots, piece;
};

HostSchedule build_schedule(long long N, int IB, int TJ, long long max_ctas, int nsm) {
    HostSchedule h;
    h.B = static_cast<int>((N + IB - 1) / IB);
    h.T = static_cast<int>((N + TJ - 1) / TJ);
    h.U = static_cast<long long>(h.B) * h.T;
    h.G = static_cast<int>(std::min<long long>(h.U, max_ctas));
    h.u0.resize(h.G + 1);
    for (int g = 0; g <= h.G; ++g) h.u0[g] = static_cast<long long>((__int128)g * h.U / h.G);
    h.first.resize(h.B);
    h.nslots.resize(h.B);
    for (int b = 0; b < h.B; ++b) {
        const long long lo = static_cast<long long>(b) * h.T;
        const long long hi = lo + h.T - 1;
        const int cf = static_cast<int>(std::upper_bound(h.u0.begin(), h.u0.end(), lo) - h.u0.begin()) - 1;
        const int cl = static_cast<int>(std::upper_bound(h.u0.begin(), h.u0.end(), hi) - h.u0.begin()) - 1;
        h.first[b] = cf;
        h.nslots[b] = cl - cf + 1;
        h.max_slots = std::max(h.max_slots, h.nslots[b]);
    }
    // Pieces differ by one unit.  The CTAs of the first (and only) wave land on SM blockIdx % #SM,
    // so CTA k, k + #SM, k + 2 #SM share an SM; when U / G resonates with #SM (N = 6000: U / G =
    // 1.27, period 3.7 = 148 / 40) the long pieces of a plain blockIdx -> piece map pile up on the
    // same SMs (6 units on some, 3 on others: 73.8 us instead of 57).  Giving the CTAs of one SM
    // consecutive pieces balances the SMs to within one unit.
    h.piece.resize(h.G);
    std::vector<int> first_of_sm(nsm + 1, 0);
    for (int sm = 0; sm < nsm; ++sm)
        first_of_sm[sm + 1] = first_of_sm[sm] + h.G / nsm + (sm < h.G % nsm ? 1 : 0);
    for (int b = 0; b < h.G; ++b) h.piece[b] = first_of_sm[b % nsm] + b / nsm;
    return h;
}

sd_status configure_w(sd_ctx* c);

// The packed one-launch kernel keeps all N records in dynamic shared memory (up to 72 KiB): the
// opt-in is per device and per function, so every context sets it for the instantiation it will
// launch, outside any stream capture, and checks the result.
sd_status set_packed_attr(sd_ctx* c) {
    if (c->precision == SD_PREC_F64 || c->N < sd::kPackedMinN || c->N > sd::kPackedMaxN) return SD_OK;
    const bool rpy = c->tensor == SD_TENSOR_RPY, kahan = c->precision != SD_PREC_F32_PLAIN, pbc = c->box > 0.0;
    const void* f = nullptr;
#define SD_PKF(T, K, P)                                                                                   \
    (c->N >= sd::kPackedWideMinN ? reinterpret_cast<const void*>(&sd::small_apply_packed_kernel<T, K, P, 512>) \
                                 : reinterpret_cast<const void*>(&sd::small_apply_packed_kernel<T, K, P>))
    if (rpy) f = kahan ? (pbc ? SD_PKF(0, true, true) : SD_PKF(0, true, false))
                       : (pbc ? SD_PKF(0, false, true) : SD_PKF(0, false, false));
    else f = kahan ? (pbc ? SD_PKF(1, true, true) : SD_PKF(1, true, false))
                   : (pbc ? SD_PKF(1, false, true) : SD_PKF(1, false, false));
#undef SD_PKF
    SD_CUDA(c, cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, sd::kPackedMaxN * 32));
    return SD_OK;
}

// Pick the kernel variant for (N, precision, tensor), build the static schedule and
// (re)allocate every scratch buffer.
sd_status configure(sd_ctx* c) {
    // the velocities of the last product survive a reconfiguration that keeps their element type
    // (sd_set_box, sd_set_tensor, sd_set_dispatch, ...): the lubrication correction needs them
    {
        int dev = -1;
        if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device)
            return fail(c, SD_ERR_INVALID_ARG, "the current CUDA device is not the one the context was created on");
    }
    // ... and so do the low words of the positions (a change of tensor, box or dispatch in the
    // middle of a run must not drop them)
    void* keep_vel = nullptr;
    void* keep_lo = nullptr;
    const size_t vel_bytes = static_cast<size_t>(c->Nrec) * 4 * elem_size(c->precision);
    if (c->vel && c->vel_bytes == vel_bytes) {
        keep_vel = c->vel;
        c->vel = nullptr;
        keep_lo = c->pos_lo;
        c->pos_lo = nullptr;
    }
    const bool lo_was_valid = c->lo_valid;
    free_buffers(c);
    c->valid = false;  // until every buffer below exists again
    c->vel = keep_vel;
    c->pos_lo = keep_lo;
    Config cfg;
    const bool f64 = c->precision == SD_PREC_F64;
    const bool rpy = c->tensor == SD_TENSOR_RPY;
    const bool pbc = c->box > 0.0;
    // where the warp-per-particle one-launch kernels stop (measured, profiles/r02_mid_n.md, sd_small.cuh): with
    // the warp-split kernel behind them at the end of the packed fp32 window (4736 in free space, 2304 in the
    // periodic box) resp. at 1000 in fp64; 2560 when only the classic tiled kernels follow
    if (c->small_user >= 0) c->small_apply_max = c->small_user;
    else if (c->jsplit == 1 || c->staging != sd::STAGE_BULK) c->small_apply_max = sd::kSmallApplyMax;
    else if (c->jsplit == 2)  // "warp-split wherever it exists": behind the 128-thread packed window
        c->small_apply_max = f64 ? sd::kW64MinN : sd::kPackedWideMinN - 1;
    else c->small_apply_max = f64 ? sd::kW64MinN : (pbc ? sd::kPackedMaxNBox : sd::kPackedMaxN);
    if (!f64) {
        const bool plain = c->precision == SD_PREC_F32_PLAIN;
        // particles per thread: 8 once there is enough work to balance 2048-particle i-blocks
        // over the SMs (more operand reuse per j record), 4 and 2 below that (measured
        // crossovers, profiles/r01e_sweep.md).  N <= small_apply_max never reaches this kernel.
        int i2 = (c->N > (pbc ? sd::kIpt8MinBox : sd::kIpt8Min)) ? 4 : (c->N > (pbc ? sd::kIpt4MinBox : sd::kIpt4Min) ? 2 : 1);
        if (c->ipt_override) i2 = c->ipt_override / 2;
        cfg.ipt = 2 * i2;
        // 2 particles per thread: 32-record tiles once there are enough of them to pay for the extra
        // slots and hand-overs (four times the work units: finer balance over 444 CTAs)
        const bool small_tiles = i2 == 1 && c->N >= sd::kTJSmallMinN && c->N <= sd::kTJSmallMaxN;
        const bool large = i2 == 4 && c->N >= sd::kRepairMaxN;  // 256-record tiles (sd_pairs_f32.cuh)
        cfg.TJ = small_tiles ? sd::kTJSmall : (large ? sd::kTJLarge : sd::kTJ);
        static const char* names[3][2][2][2] = {
            {{{"pairs_f32x2_i2_rpy_kahan", "pairs_f32x2_i2_rpy_kahan_pbc"},
              {"pairs_f32x2_i2_rpy_plain", "pairs_f32x2_i2_rpy_plain_pbc"}},
             {{"pairs_f32x2_i2_oseen_kahan", "pairs_f32x2_i2_oseen_kahan_pbc"},
              {"pairs_f32x2_i2_oseen_plain", "pairs_f32x2_i2_oseen_plain_pbc"}}},
            {{{"pairs_f32x2_i4_rpy_kahan", "pairs_f32x2_i4_rpy_kahan_pbc"},
              {"pairs_f32x2_i4_rpy_plain", "pairs_f32x2_i4_rpy_plain_pbc"}},
             {{"pairs_f32x2_i4_oseen_kahan", "pairs_f32x2_i4_oseen_kahan_pbc"},
              {"pairs_f32x2_i4_oseen_plain", "pairs_f32x2_i4_oseen_plain_pbc"}}},
            {{{"pairs_f32x2_i8_rpy_kahan", "pairs_f32x2_i8_rpy_kahan_pbc"},
              {"pairs_f32x2_i8_rpy_plain", "pairs_f32x2_i8_rpy_plain_pbc"}},
             {{"pairs_f32x2_i8_oseen_kahan", "pairs_f32x2_i8_oseen_kahan_pbc"},
              {"pairs_f32x2_i8_oseen_plain", "pairs_f32x2_i8_oseen_plain_pbc"}}}};
        cfg.name = names[i2 == 4 ? 2 : (i2 == 2 ? 1 : 0)][rpy ? 0 : 1][plain ? 1 : 0][pbc ? 1 : 0];
        if (large)
            cfg.kernel = pbc ? f32_pick_large<true>(rpy, plain) : f32_pick_large<false>(rpy, plain);
        else if (i2 == 4)
            cfg.kernel = pbc ? f32_pick<4, true>(rpy, plain) : f32_pick<4, false>(rpy, plain);
        else if (i2 == 2)
            cfg.kernel = pbc ? f32_pick<2, true>(rpy, plain) : f32_pick<2, false>(rpy, plain);
        else if (small_tiles)
            cfg.kernel = pbc ? f32_pick<1, true, sd::kTJSmall>(rpy, plain) : f32_pick<1, false, sd::kTJSmall>(rpy, plain);
        else
            cfg.kernel = pbc ? f32_pick<1, true>(rpy, plain) : f32_pick<1, false>(rpy, plain);
        if (c->staging != sd::STAGE_BULK) {  // ablation variants: RPY, Kahan, free space only
            if (!rpy || plain || pbc)
                return fail(c, SD_ERR_UNSUPPORTED,
                            "staging ablation exists for RPY, fp32-Kahan, free space only: call sd_set_staging(ctx, 0) first");
            const bool naive = c->staging == sd::STAGE_NAIVE;
#define SD_STAGED_R(I2V, TJV, RV)                                                                   \
    (naive ? reinterpret_cast<const void*>(&sd::pairs_f32_kernel<I2V, 0, 0, false, sd::STAGE_NAIVE, TJV, RV>) \
           : reinterpret_cast<const void*>(&sd::pairs_f32_kernel<I2V, 0, 0, false, sd::STAGE_SYNC, TJV, RV>))
#define SD_STAGED_T(I2V, TJV) SD_STAGED_R(I2V, TJV, 1)
#define SD_STAGED(I2V) SD_STAGED_T(I2V, sd::kTJ)
            // same repair variant as the bulk-copy kernel of this size: the modes stay bit-identical
            cfg.kernel = (i2 == 4) ? (large ? SD_STAGED_R(4, sd::kTJLarge, 0) : SD_STAGED(4))
                                   : ((i2 == 2) ? SD_STAGED(2)
                                                : (small_tiles ? SD_STAGED_T(1, sd::kTJSmall) : SD_STAGED(1)));
#undef SD_STAGED_R
#undef SD_STAGED_T
#undef SD_STAGED
            static const char* snames[2][3] = {
                {"pairs_f32x2_i2_rpy_kahan_naive", "pairs_f32x2_i4_rpy_kahan_naive", "pairs_f32x2_i8_rpy_kahan_naive"},
                {"pairs_f32x2_i2_rpy_kahan_sync", "pairs_f32x2_i4_rpy_kahan_sync", "pairs_f32x2_i8_rpy_kahan_sync"}};
            cfg.name = snames[naive ? 0 : 1][i2 == 4 ? 2 : (i2 == 2 ? 1 : 0)];
        }
    } else {
        // 4 particles per thread (one CTA per SM) once 1024-particle i-blocks balance over the
        // SMs: one LDS.128 per pair instead of two; 2 and 1 below (measured crossovers)
        if (c->staging != sd::STAGE_BULK)
            return fail(c, SD_ERR_UNSUPPORTED,
                        "staging ablation exists for RPY, fp32-Kahan, free space only: call sd_set_staging(ctx, 0) first");
        cfg.ipt = (c->N > sd::kIpt4Min64) ? 4 : (c->N > sd::kIpt2Min64 ? 2 : 1);
        if (c->ipt_override) cfg.ipt = std::max(1, c->ipt_override / 2);
        const bool large64 = cfg.ipt == 4 && c->N >= sd::kRepairMaxN;  // 128-record tiles (sd_pairs_f64.cuh)
        cfg.TJ = large64 ? sd::kTJ64Large : sd::kTJ64;
        static const char* names64[3][2][2] = {
            {{"pairs_f64_i1_rpy", "pairs_f64_i1_rpy_pbc"}, {"pairs_f64_i1_oseen", "pairs_f64_i1_oseen_pbc"}},
            {{"pairs_f64_i2_rpy", "pairs_f64_i2_rpy_pbc"}, {"pairs_f64_i2_oseen", "pairs_f64_i2_oseen_pbc"}},
            {{"pairs_f64_i4_rpy", "pairs_f64_i4_rpy_pbc"}, {"pairs_f64_i4_oseen", "pairs_f64_i4_oseen_pbc"}}};
        cfg.name = names64[cfg.ipt == 4 ? 2 : (cfg.ipt == 2 ? 1 : 0)][rpy ? 0 : 1][pbc ? 1 : 0];
        if (large64)
            cfg.kernel = pbc ? f64_pick<4, true, sd::kTJ64Large>(rpy) : f64_pick<4, false, sd::kTJ64Large>(rpy);
        else if (cfg.ipt == 4)
            cfg.kernel = pbc ? f64_pick<4, true>(rpy) : f64_pick<4, false>(rpy);
        else if (cfg.ipt == 2)
            cfg.kernel = pbc ? f64_pick<2, true>(rpy) : f64_pick<2, false>(rpy);
        else
            cfg.kernel = pbc ? f64_pick<1, true>(rpy) : f64_pick<1, false>(rpy);
    }
    cfg.IB = sd::kThreads * cfg.ipt;
    int occ = 0;
    SD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, cfg.kernel, sd::kThreads, 0));
    if (occ < 1) return fail(c, SD_ERR_CUDA, "pair kernel does not fit on an SM");
    const HostSchedule hs = build_schedule(c->N, cfg.IB, cfg.TJ, static_cast<long long>(c->num_sms) * occ, c->num_sms);
    cfg.B = hs.B, cfg.T = hs.T, cfg.U = hs.U, cfg.G = hs.G, cfg.max_slots = hs.max_slots;
    const std::vector<long long>& u0 = hs.u0;
    const std::vector<int>&first = hs.first, &nslots = hs.nslots, &piece = hs.piece;
    c->cfg = cfg;

    const size_t es = elem_size(c->precision);
    const size_t v4 = 4 * es;
    const size_t nrec = static_cast<size_t>(c->Nrec);
    SD_CUDA(c, cudaMalloc(&c->rec, nrec * 2 * v4));
    const size_t part_per_slot = f64 ? nrec * v4 : nrec * 2 * v4;
    SD_CUDA(c, cudaMalloc(&c->part, part_per_slot * cfg.max_slots));
    if (!c->vel) {  // "velocities of the previous step" start at zero (cold start of the lubrication loop)
        SD_CUDA(c, cudaMalloc(&c->vel, nrec * v4));
        SD_CUDA(c, cudaMemset(c->vel, 0, nrec * v4));
        c->vel_bytes = nrec * v4;
    }
    const bool fresh_lo = c->pos_lo == nullptr;
    if (fresh_lo) SD_CUDA(c, cudaMalloc(&c->pos_lo, nrec * v4));
    SD_CUDA(c, cudaMalloc(&c->pos_half, nrec * v4));
    SD_CUDA(c, cudaMalloc(&c->pos_alt, nrec * v4));
    SD_CUDA(c, cudaMalloc(&c->force_buf, nrec * v4));
    if (fresh_lo) SD_CUDA(c, cudaMemset(c->pos_lo, 0, nrec * v4));
    SD_CUDA(c, cudaMalloc(&c->d_cta_u0, sizeof(long long) * (cfg.G + 1)));
    SD_CUDA(c, cudaMalloc(&c->d_blk_first, sizeof(int) * cfg.B));
    SD_CUDA(c, cudaMalloc(&c->d_blk_nslots, sizeof(int) * cfg.B));
    SD_CUDA(c, cudaMalloc(&c->d_cta_piece, sizeof(int) * cfg.G));
    SD_CUDA(c, cudaMemcpy(c->d_cta_piece, piece.data(), sizeof(int) * cfg.G, cudaMemcpyHostToDevice));
    SD_CUDA(c, cudaMemcpy(c->d_cta_u0, u0.data(), sizeof(long long) * (cfg.G + 1), cudaMemcpyHostToDevice));
    SD_CUDA(c, cudaMemcpy(c->d_blk_first, first.data(), sizeof(int) * cfg.B, cudaMemcpyHostToDevice));
    SD_CUDA(c, cudaMemcpy(c->d_blk_nslots, nslots.data(), sizeof(int) * cfg.B, cudaMemcpyHostToDevice));
    c->lo_valid = fresh_lo ? true : lo_was_valid;  // fresh words are zero; kept ones keep their state
    // mid N in the fp32 modes: the whole product in one launch of the warp-split kernel
    const long long wmax = f64 ? sd::kW64MaxN : (pbc ? sd::kWMaxNBox : sd::kWMaxN);
    if (c->staging == sd::STAGE_BULK && c->N > c->small_apply_max &&
        (c->jsplit == 2 || (c->jsplit == 0 && c->N <= wmax))) {
        sd_status ws = configure_w(c);
        if (ws != SD_OK) return ws;
    }
    {
        sd_status ps = set_packed_attr(c);
        if (ps != SD_OK) return ps;
    }
    c->valid = true;
    return SD_OK;
}

// ---- warp-split one-launch kernel (sd_pairs_f32w.cuh) -----------------------------------------
template <int I2>
const void* w_pick(bool rpy, bool plain, bool pbc) {
#define SD_W(T, A, P) reinterpret_cast<const void*>(&sd::pairs_f32w_kernel<I2, T, A, P>)
    if (rpy) {
        if (plain) return pbc ? SD_W(0, 1, true) : SD_W(0, 1, false);
        return pbc ? SD_W(0, 0, true) : SD_W(0, 0, false);
    }
    if (plain) return pbc ? SD_W(1, 1, true) : SD_W(1, 1, false);
    return pbc ? SD_W(1, 0, true) : SD_W(1, 0, false);
#undef SD_W
}

sd_status configure_w(sd_ctx* c) {
    const bool rpy = c->tensor == SD_TENSOR_RPY, plain = c->precision == SD_PREC_F32_PLAIN, pbc = c->box > 0.0;
    const bool f64 = c->precision == SD_PREC_F64;
    Config w;
    size_t smem = 0;
    w.TJ = sd::kWQ;  // the schedule is cut at 4-record granularity; tiles are private to the warps
    if (f64) {
        w.ipt = 4;
        w.IB = 32 * 4;
#define SD_W64(T, P) reinterpret_cast<const void*>(&sd::pairs_f64w_kernel<4, T, P>)
        w.kernel = rpy ? (pbc ? SD_W64(0, true) : SD_W64(0, false)) : (pbc ? SD_W64(1, true) : SD_W64(1, false));
#undef SD_W64
        smem = sd::W64Shape<4>::smem_bytes;
    } else {
        w.ipt = 8;
        w.IB = 64 * 4;
        w.kernel = w_pick<4>(rpy, plain, pbc);
        smem = sd::WShape<4>::smem_bytes;
    }
    static const char* wn[2][2][2] = {{{"pairs_f32x2_w8_rpy_kahan", "pairs_f32x2_w8_rpy_kahan_pbc"},
                                       {"pairs_f32x2_w8_rpy_plain", "pairs_f32x2_w8_rpy_plain_pbc"}},
                                      {{"pairs_f32x2_w8_oseen_kahan", "pairs_f32x2_w8_oseen_kahan_pbc"},
                                       {"pairs_f32x2_w8_oseen_plain", "pairs_f32x2_w8_oseen_plain_pbc"}}};
    w.name = wn[rpy ? 0 : 1][plain ? 1 : 0][pbc ? 1 : 0];
    static const char* wn64[2][2] = {{"pairs_f64_w4_rpy", "pairs_f64_w4_rpy_pbc"}, {"pairs_f64_w4_oseen", "pairs_f64_w4_oseen_pbc"}};
    if (f64) w.name = wn64[rpy ? 0 : 1][pbc ? 1 : 0];
    SD_CUDA(c, cudaFuncSetAttribute(w.kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    int occ = 0;
    SD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, w.kernel, sd::kThreads, smem));
    if (occ < 1) return fail(c, SD_ERR_CUDA, "warp-split pair kernel does not fit on an SM");
    // one CTA per SM (the kernel takes piece = blockIdx.x and recomputes the cut points g U / G)
    const HostSchedule hs = build_schedule(c->N, w.IB, w.TJ, c->num_sms, c->num_sms);
    w.B = hs.B, w.T = hs.T, w.U = hs.U, w.G = hs.G, w.max_slots = hs.max_slots;
    c->wcfg = w;
    c->w_smem = smem;
    const size_t nrec = static_cast<size_t>(c->Nrec);
    SD_CUDA(c, cudaMalloc(&c->w_part, nrec * (f64 ? sizeof(double4) : 2 * sizeof(float4)) * w.max_slots));
    SD_CUDA(c, cudaMalloc(&c->w_blk_done, sizeof(int) * w.B));
    SD_CUDA(c, cudaMemset(c->w_blk_done, 0, sizeof(int) * w.B));
    SD_CUDA(c, cudaMalloc(&c->w_cta_u0, sizeof(long long) * (w.G + 1)));
    SD_CUDA(c, cudaMalloc(&c->w_blk_first, sizeof(int) * w.B));
    SD_CUDA(c, cudaMalloc(&c->w_blk_nslots, sizeof(int) * w.B));
    SD_CUDA(c, cudaMalloc(&c->w_cta_piece, sizeof(int) * w.G));
    SD_CUDA(c, cudaMemcpy(c->w_cta_u0, hs.u0.data(), sizeof(long long) * (w.G + 1), cudaMemcpyHostToDevice));
    SD_CUDA(c, cudaMemcpy(c->w_blk_first, hs.first.data(), sizeof(int) * w.B, cudaMemcpyHostToDevice));
    SD_CUDA(c, cudaMemcpy(c->w_blk_nslots, hs.nslots.data(), sizeof(int) * w.B, cudaMemcpyHostToDevice));
    SD_CUDA(c, cudaMemcpy(c->w_cta_piece, hs.piece.data(), sizeof(int) * w.G, cudaMemcpyHostToDevice));
    if (f64) {
        std::vector<double4> pad(2 * sd::kW64SJ, make_double4(0.0, 0.0, 0.0, 0.0));
        for (int q = 0; q < sd::kW64SJ; ++q) pad[q] = make_double4(SD_PAD_POS, SD_PAD_POS, SD_PAD_POS, 0.0);
        SD_CUDA(c, cudaMalloc(&c->w_pad, pad.size() * sizeof(double4)));
        SD_CUDA(c, cudaMemcpy(c->w_pad, pad.data(), pad.size() * sizeof(double4), cudaMemcpyHostToDevice));
    } else {
        std::vector<float4> pad(2 * sd::kWSJ, make_float4(0.f, 0.f, 0.f, 0.f));
        for (int q = 0; q < sd::kWSJ; ++q) pad[q] = make_float4(SD_PAD_POS, SD_PAD_POS, SD_PAD_POS, 0.f);
        SD_CUDA(c, cudaMalloc(&c->w_pad, pad.size() * sizeof(float4)));
        SD_CUDA(c, cudaMemcpy(c->w_pad, pad.data(), pad.size() * sizeof(float4), cudaMemcpyHostToDevice));
    }
    SD_CUDA(c, cudaMalloc(&c->grav_buf, nrec * 4 * elem_size(c->precision)));
    c->w_on = true;
    return SD_OK;
}

sd::Schedule schedule_of(const sd_ctx* c) {
    sd::Schedule s;
    s.cta_u0 = c->d_cta_u0;
    s.blk_first_cta = c->d_blk_first;
    s.blk_nslots = c->d_blk_nslots;
    s.cta_piece = c->d_cta_piece;
    s.T = c->cfg.T;
    s.B = c->cfg.B;
    s.G = c->cfg.G;
    return s;
}

sd_status check_launch(sd_ctx* c, const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(c, SD_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
    ++c->launches;
    return SD_OK;
}

sd_status launch_pack(sd_ctx* c, const void* pos, const void* force, int what, const double g[3],
                      cudaStream_t st) {
    const int n = static_cast<int>(c->N), nrec = static_cast<int>(c->Nrec);
    const int blocks = (nrec + 255) / 256;
    const double gx = g ? g[0] : 0.0, gy = g ? g[1] : 0.0, gz = g ? g[2] : 0.0;
    const double c1 = c->mu0 * 0.75 * c->a;  // folded into the force lane of the records
    if (c->precision == SD_PREC_F64)
        sd::pack_kernel<double4><<<blocks, 256, 0, st>>>(
            static_cast<const double4*>(pos), static_cast<const double4*>(force),
            static_cast<double4*>(c->rec), what, gx, gy, gz, c1, n, nrec);
    else
        sd::pack_kernel<float4><<<blocks, 256, 0, st>>>(
            static_cast<const float4*>(pos), static_cast<const float4*>(force),
            static_cast<float4*>(c->rec), what, gx, gy, gz, c1, n, nrec);
    return check_launch(c, "pack_kernel");
}

sd_status launch_pairs_impl(sd_ctx* c, cudaStream_t st);

// nearest-image constants (PAPER.md:115 footnote 1): L is rounded to S first, 1/L is the
// correctly rounded quotient in S (reading B2); free space: all zero
template <typename S>
void box_coef(const sd_ctx* c, S& invL, S& mL, S& magic) {
    invL = mL = magic = S(0);
    if (c->box > 0.0) {
        const S L = static_cast<S>(c->box);
        invL = S(1) / L;
        mL = -L;
        magic = (sizeof(S) == 4) ? static_cast<S>(12582912.0) : static_cast<S>(6755399441055744.0);
    }
}

// coefficients in the folded units of sd_common.cuh (PairCoefT): they depend on a only
template <typename S>
sd::PairCoefT<S> folded_coef(const sd_ctx* c) {
    const double a = c->a;
    sd::PairCoefT<S> k;
    k.k2 = static_cast<S>(2.0 * a * a / 3.0);
    k.m3k2 = static_cast<S>(-2.0 * a * a);
    k.mu0r = static_cast<S>(4.0 / (3.0 * a));
    k.ovA = static_cast<S>(-3.0 / (8.0 * a * a));
    k.ovB = static_cast<S>(1.0 / (8.0 * a * a));
    k.thr = (c->tensor == SD_TENSOR_RPY) ? static_cast<S>(4.0 * a * a) : static_cast<S>(1e-30);
    k.clampv = static_cast<S>(4.0 * a * a);
    box_coef<S>(c, k.invL, k.mL, k.magic);
    return k;
}

// runs `impl` (a pair-kernel launch); while profiling is on, between two events on the stream
template <typename Impl>
sd_status profiled(sd_ctx* c, cudaStream_t st, Impl impl) {
    if (!c->profiling || c->prof_events.size() >= 4096) return impl();
    std::pair<cudaEvent_t, cudaEvent_t> ev;
    if (!c->prof_pool.empty()) {
        ev = c->prof_pool.back();
        c->prof_pool.pop_back();
    } else {
        SD_CUDA(c, cudaEventCreate(&ev.first));
        SD_CUDA(c, cudaEventCreate(&ev.second));
    }
    SD_CUDA(c, cudaEventRecord(ev.first, st));
    sd_status s = impl();
    SD_CUDA(c, cudaEventRecord(ev.second, st));
    c->prof_events.push_back(ev);
    return s;
}

sd_status launch_pairs(sd_ctx* c, cudaStream_t st) {
    return profiled(c, st, [&]() { return launch_pairs_impl(c, st); });
}

// one product (+ fused update) in one launch of the warp-split kernel; arguments as launch_small_apply
sd_status launch_w(sd_ctx* c, const void* posx, const void* force, void* vel, const void* pos_base,
                   void* pos_out, double dt, int mode, cudaStream_t st) {
    return profiled(c, st, [&]() -> sd_status {
        if (c->precision == SD_PREC_F64) {
            sd::Schedule sch;
            sch.cta_u0 = c->w_cta_u0, sch.blk_first_cta = c->w_blk_first, sch.blk_nslots = c->w_blk_nslots;
            sch.cta_piece = c->w_cta_piece;
            sch.T = c->wcfg.T, sch.B = c->wcfg.B, sch.G = c->wcfg.G;
            sd::PairCoef64 k = folded_coef<double>(c);
            float thr = (c->tensor == SD_TENSOR_RPY) ? static_cast<float>(4.0 * c->a * c->a * (1.0 + 1e-6)) : 1e-30f;
            sd::FinArgs64 fin;
            fin.vel = static_cast<double4*>(vel);
            fin.pos_base = static_cast<const double4*>(pos_base);
            fin.pos_out = static_cast<double4*>(pos_out);
            fin.dt = dt, fin.c1 = c->mu0 * 0.75 * c->a, fin.mu0 = c->mu0, fin.mode = mode;
            const double4* pp = static_cast<const double4*>(posx);
            const double4* ff = static_cast<const double4*>(force);
            const double4* pad = static_cast<const double4*>(c->w_pad);
            double4* part = static_cast<double4*>(c->w_part);
            int n = static_cast<int>(c->N);
            long long stride = c->Nrec;
            void* args[] = {&pp, &ff, &pad, &part, &c->w_blk_done, &sch, &k, &thr, &fin, &n, &stride};
            cudaError_t e = cudaLaunchKernel(c->wcfg.kernel, dim3(c->wcfg.G), dim3(sd::kThreads), args, c->w_smem, st);
            if (e != cudaSuccess) return fail(c, SD_ERR_CUDA, std::string("pairs_f64w: ") + cudaGetErrorString(e));
            return check_launch(c, c->wcfg.name);
        }
        sd::Schedule sch;
        sch.cta_u0 = c->w_cta_u0;
        sch.blk_first_cta = c->w_blk_first;
        sch.blk_nslots = c->w_blk_nslots;
        sch.cta_piece = c->w_cta_piece;
        sch.T = c->wcfg.T, sch.B = c->wcfg.B, sch.G = c->wcfg.G;
        sd::PairCoef k = folded_coef<float>(c);
        sd::FinArgs fin;
        fin.vel = static_cast<float4*>(vel);
        fin.pos_base = static_cast<const float4*>(pos_base);
        fin.pos_lo = static_cast<float4*>(c->pos_lo);
        fin.pos_out = static_cast<float4*>(pos_out);
        fin.dt = dt;
        fin.c1 = c->mu0 * 0.75 * c->a;
        fin.mu0 = c->mu0;
        fin.mode = mode;
        fin.pos_comp = c->pos_comp;
        const float4* pp = static_cast<const float4*>(posx);
        const float4* ff = static_cast<const float4*>(force);
        const float4* pad = static_cast<const float4*>(c->w_pad);
        float4* part = static_cast<float4*>(c->w_part);
        int n = static_cast<int>(c->N);
        long long stride = c->Nrec;
        void* args[] = {&pp, &ff, &pad, &part, &c->w_blk_done, &sch, &k, &fin, &n, &stride};
        cudaError_t e = cudaLaunchKernel(c->wcfg.kernel, dim3(c->wcfg.G), dim3(sd::kThreads), args, c->w_smem, st);
        if (e != cudaSuccess) return fail(c, SD_ERR_CUDA, std::string("pairs_f32w: ") + cudaGetErrorString(e));
        return check_launch(c, c->wcfg.name);
    });
}

sd_status launch_pairs_impl(sd_ctx* c, cudaStream_t st) {
    sd::Schedule sch = schedule_of(c);
    int n = static_cast<int>(c->N);
    long long stride = c->Nrec;
    if (c->precision == SD_PREC_F64) {
        sd::PairCoef64 k = folded_coef<double>(c);
        // threshold on the fp32 copy of r^2, inflated so that rounding can only send a pair to
        // the exact path, never keep an overlapping one on the fast path
        float thr = (c->tensor == SD_TENSOR_RPY) ? static_cast<float>(4.0 * c->a * c->a * (1.0 + 1e-6)) : 1e-30f;
        const double4* rec = static_cast<const double4*>(c->rec);
        double4* part = static_cast<double4*>(c->part);
        void* args[] = {&rec, &part, &sch, &k, &thr, &n, &stride};
        cudaError_t e = cudaLaunchKernel(c->cfg.kernel, dim3(c->cfg.G), dim3(sd::kThreads), args, 0, st);
        if (e != cudaSuccess) return fail(c, SD_ERR_CUDA, std::string("pairs_f64: ") + cudaGetErrorString(e));
    } else {
        sd::PairCoef k = folded_coef<float>(c);
        const float4* rec = static_cast<const float4*>(c->rec);
        float4* part = static_cast<float4*>(c->part);
        void* args[] = {&rec, &part, &sch, &k, &n, &stride};
        cudaError_t e = cudaLaunchKernel(c->cfg.kernel, dim3(c->cfg.G), dim3(sd::kThreads), args, 0, st);
        if (e != cudaSuccess) return fail(c, SD_ERR_CUDA, std::string("pairs_f32: ") + cudaGetErrorString(e));
    }
    return check_launch(c, c->cfg.name);
}

template <int MODE>
sd_status launch_finalize(sd_ctx* c, void* vel, void* pos, double dt, cudaStream_t st) {
    const int n = static_cast<int>(c->N);
    const int blocks = (n + sd::kFinThreads - 1) / sd::kFinThreads;
    if (c->precision == SD_PREC_F64)
        sd::finalize_f64_kernel<MODE><<<blocks, sd::kFinThreads, 0, st>>>(
            static_cast<const double4*>(c->part), c->d_blk_nslots, static_cast<double4*>(c->rec),
            static_cast<double4*>(vel), static_cast<double4*>(pos),
            static_cast<double4*>(c->pos_half), dt, 4.0 / (3.0 * c->a), n, c->cfg.IB, c->Nrec,
            c->tensor, 4.0 * c->a * c->a, 2.0 * c->a * c->a / 3.0);
    else
        sd::finalize_f32_kernel<MODE><<<blocks, sd::kFinThreads, 0, st>>>(
            static_cast<const float4*>(c->part), c->d_blk_nslots, static_cast<float4*>(c->rec),
            static_cast<float4*>(vel), static_cast<float4*>(pos), static_cast<float4*>(c->pos_lo),
            static_cast<float4*>(c->pos_half), dt, 4.0 / (3.0 * c->a), n, c->cfg.IB, c->Nrec,
            c->pos_comp, c->tensor, static_cast<float>(4.0 * c->a * c->a),
            static_cast<float>(2.0 * c->a * c->a / 3.0));
    return check_launch(c, "finalize_kernel");
}

// ---- small-N path (sd_small.cuh) -------------------------------------------------------------
template <typename S>
sd::CoefT<S> coef_of(const sd_ctx* c) {
    const double a = c->a, mu0 = c->mu0;
    sd::CoefT<S> k;
    k.c1 = static_cast<S>(mu0 * 0.75 * a);
    k.c2 = static_cast<S>(mu0 * 0.5 * a * a * a);
    k.m3c2 = static_cast<S>(-1.5 * mu0 * a * a * a);
    k.mu0 = static_cast<S>(mu0);
    k.ovA = static_cast<S>(-9.0 * mu0 / (32.0 * a));
    k.ovB = static_cast<S>(3.0 * mu0 / (32.0 * a));
    k.four_a2 = static_cast<S>(4.0 * a * a);
    box_coef<S>(c, k.invL, k.mL, k.magic);
    return k;
}

template <typename T4, bool KAHAN>
sd_status launch_small_apply_t(sd_ctx* c, const void* posx, const void* force, const double g[3],
                               void* vel, const void* pos_base, void* pos_out, double dt, int mode,
                               cudaStream_t st) {
    typedef typename sd::Vec4<T4>::S S;
    const int n = static_cast<int>(c->N);
    const int ipw = (n > 2368) ? 2 : 1;  // one particle per warp while that leaves SMs idle
    const int per_cta = (sd::kSmallThreads / 32) * ipw;
    const int blocks = (n + per_cta - 1) / per_cta;
    const sd::CoefT<S> k = coef_of<S>(c);
    const double gx = g ? g[0] : 0.0, gy = g ? g[1] : 0.0, gz = g ? g[2] : 0.0;
    const bool rpy = c->tensor == SD_TENSOR_RPY;
#define SD_SMALL_LAUNCH(TEN, IPW)                                                                  \
    sd::small_apply_kernel<T4, TEN, KAHAN, IPW><<<blocks, sd::kSmallThreads, 0, st>>>(             \
        static_cast<const T4*>(posx), static_cast<const T4*>(force), gx, gy, gz,                   \
        static_cast<T4*>(vel), static_cast<const T4*>(pos_base), static_cast<T4*>(c->pos_lo),      \
        static_cast<T4*>(pos_out), dt, mode, k, n, c->pos_comp)
    if (rpy) {
        if (ipw == 2) SD_SMALL_LAUNCH(0, 2); else SD_SMALL_LAUNCH(0, 1);
    } else {
        if (ipw == 2) SD_SMALL_LAUNCH(1, 2); else SD_SMALL_LAUNCH(1, 1);
    }
#undef SD_SMALL_LAUNCH
    return check_launch(c, "small_apply_kernel");
}

// fp32 modes from kPackedMinN particles on: the packed variant (sd_small.cuh)
template <int TENSOR, bool KAHAN, bool PBC>
void launch_small_packed_k(sd_ctx* c, const void* posx, const void* force, const double g[3], void* vel,
                           const void* pos_base, void* pos_out, double dt, int mode, cudaStream_t st) {
    const int n = static_cast<int>(c->N);
    const int threads = sd::packed_threads(n);
    const int per_cta = (threads / 32) * 2;
    const int blocks = (n + per_cta - 1) / per_cta;
    const double gx = g ? g[0] : 0.0, gy = g ? g[1] : 0.0, gz = g ? g[2] : 0.0;
    const size_t smem = static_cast<size_t>(n) * 32;  // opt-in above 48 KiB: set_packed_attr, at configure time
#define SD_PK_ARGS                                                                                        \
    static_cast<const float4*>(posx), static_cast<const float4*>(force), gx, gy, gz,                       \
        static_cast<float4*>(vel), static_cast<const float4*>(pos_base), static_cast<float4*>(c->pos_lo),  \
        static_cast<float4*>(pos_out), dt, mode, folded_coef<float>(c), c->mu0 * 0.75 * c->a, c->mu0, n,   \
        c->pos_comp
    if (threads == 512)
        sd::small_apply_packed_kernel<TENSOR, KAHAN, PBC, 512><<<blocks, 512, smem, st>>>(SD_PK_ARGS);
    else
        sd::small_apply_packed_kernel<TENSOR, KAHAN, PBC><<<blocks, sd::kPackedThreads, smem, st>>>(SD_PK_ARGS);
#undef SD_PK_ARGS
}
template <bool KAHAN>
sd_status launch_small_packed(sd_ctx* c, const void* posx, const void* force, const double g[3], void* vel,
                              const void* pos_base, void* pos_out, double dt, int mode, cudaStream_t st) {
    const bool rpy = c->tensor == SD_TENSOR_RPY, pbc = c->box > 0.0;
#define SD_PK(T, P) launch_small_packed_k<T, KAHAN, P>(c, posx, force, g, vel, pos_base, pos_out, dt, mode, st)
    if (rpy) { if (pbc) SD_PK(0, true); else SD_PK(0, false); }
    else { if (pbc) SD_PK(1, true); else SD_PK(1, false); }
#undef SD_PK
    return check_launch(c, "small_apply_packed_kernel");
}

sd_status launch_small_apply(sd_ctx* c, const void* posx, const void* force, const double g[3],
                             void* vel, const void* pos_base, void* pos_out, double dt, int mode,
                             cudaStream_t st) {
    if (c->w_on)  // mid N: warp-split kernel; a uniform force has been written to grav_buf by the caller
        return launch_w(c, posx, force ? force : c->grav_buf, vel, pos_base, pos_out, dt, mode, st);
    if (c->precision != SD_PREC_F64 && c->N >= sd::kPackedMinN && c->N <= sd::kPackedMaxN &&
        c->N <= c->small_apply_max) {
        if (c->precision == SD_PREC_F32_PLAIN)
            return launch_small_packed<false>(c, posx, force, g, vel, pos_base, pos_out, dt, mode, st);
        return launch_small_packed<true>(c, posx, force, g, vel, pos_base, pos_out, dt, mode, st);
    }
    if (c->precision == SD_PREC_F64)
        return launch_small_apply_t<double4, false>(c, posx, force, g, vel, pos_base, pos_out, dt, mode, st);
    if (c->precision == SD_PREC_F32_PLAIN)
        return launch_small_apply_t<float4, false>(c, posx, force, g, vel, pos_base, pos_out, dt, mode, st);
    return launch_small_apply_t<float4, true>(c, posx, force, g, vel, pos_base, pos_out, dt, mode, st);
}

template <typename T4, bool KAHAN>
sd_status launch_stepper_t(sd_ctx* c, void* pos, const void* force, const double g[3], double dt,
                           long long n_steps, int integrator, cudaStream_t st) {
    typedef typename sd::Vec4<T4>::S S;
    const int n = static_cast<int>(c->N);
    const int sub = (n <= 32) ? 32 : 16;  // lanes per particle; n <= kStepperMax = 64
    const int threads = (n * sub + 31) / 32 * 32;
    const sd::CoefT<S> k = coef_of<S>(c);
    const double gx = g ? g[0] : 0.0, gy = g ? g[1] : 0.0, gz = g ? g[2] : 0.0;
    const bool rpy = c->tensor == SD_TENSOR_RPY;
    // bounded launches: a kernel that runs for minutes is a hazard on shared boxes
    const long long chunk = 1LL << 20;
    for (long long done = 0; done < n_steps; done += chunk) {
        const long long ns = std::min(chunk, n_steps - done);
#define SD_STEP_LAUNCH(TEN, SUB)                                                                   \
    sd::small_stepper_kernel<T4, TEN, KAHAN, SUB><<<1, threads, 0, st>>>(                          \
        static_cast<T4*>(pos), static_cast<T4*>(c->pos_lo), static_cast<const T4*>(force), gx, gy, \
        gz, static_cast<T4*>(c->vel), dt, ns, integrator, k, n, c->pos_comp)
        if (rpy) {
            if (sub == 32) SD_STEP_LAUNCH(0, 32); else SD_STEP_LAUNCH(0, 16);
        } else {
            if (sub == 32) SD_STEP_LAUNCH(1, 32); else SD_STEP_LAUNCH(1, 16);
        }
#undef SD_STEP_LAUNCH
        sd_status s = check_launch(c, "small_stepper_kernel");
        if (s != SD_OK) return s;
    }
    return SD_OK;
}

sd_status launch_stepper(sd_ctx* c, void* pos, const void* force, const double g[3], double dt,
                         long long n_steps, int integrator, cudaStream_t st) {
    if (c->precision == SD_PREC_F64)
        return launch_stepper_t<double4, false>(c, pos, force, g, dt, n_steps, integrator, st);
    if (c->precision == SD_PREC_F32_PLAIN)
        return launch_stepper_t<float4, false>(c, pos, force, g, dt, n_steps, integrator, st);
    return launch_stepper_t<float4, true>(c, pos, force, g, dt, n_steps, integrator, st);
}

// cell-grid scratch of the lubrication step (allocated on first use, never inside a stream capture)
sd_status ensure_lub_buffers(sd_ctx* c) {
    const int n = static_cast<int>(c->N);
    unsigned H = 512;  // 2^(3 bits) buckets, at least one per particle
    while (H < static_cast<unsigned>(n)) H <<= 3;
    c->lub_H = H;
    // every buffer on its own: after a failed allocation the next call allocates what is missing
    if (!c->lub_spos) SD_CUDA(c, cudaMalloc(&c->lub_spos, 4 * elem_size(c->precision) * n));
    if (!c->lub_svel) SD_CUDA(c, cudaMalloc(&c->lub_svel, 4 * elem_size(c->precision) * n));
    if (!c->lub_bucket) SD_CUDA(c, cudaMalloc(&c->lub_bucket, sizeof(unsigned) * n));
    if (!c->lub_count) {  // zeroed once here; every call leaves it zeroed (lub_gather_kernel)
        SD_CUDA(c, cudaMalloc(&c->lub_count, sizeof(unsigned) * (H + 1)));
        SD_CUDA(c, cudaMemset(c->lub_count, 0, sizeof(unsigned) * (H + 1)));
        c->lub_count_dirty = false;
    }
    if (!c->lub_start) SD_CUDA(c, cudaMalloc(&c->lub_start, sizeof(unsigned) * (H + 1)));
    if (!c->lub_cursor) SD_CUDA(c, cudaMalloc(&c->lub_cursor, sizeof(unsigned) * H));
    if (!c->lub_order) SD_CUDA(c, cudaMalloc(&c->lub_order, sizeof(int) * n));
    if (!c->lub_slots) SD_CUDA(c, cudaMalloc(&c->lub_slots, sizeof(int2) * n));
    if (!c->lub_tmp) {  // block totals of the two-launch scan
        c->lub_tmp_bytes = sizeof(unsigned) * ((H + 1 + sd::kScanBlock - 1) / sd::kScanBlock);
        SD_CUDA(c, cudaMalloc(&c->lub_tmp, c->lub_tmp_bytes));
    }
    return SD_OK;
}

// force_out = F^ext - C(pos, vel)  (sd_lub.cuh).  fext NULL: uniform force g.
sd_status launch_lubrication(sd_ctx* c, const void* pos, const void* vel, const void* fext,
                             const double g[3], void* force_out, cudaStream_t st) {
    const int n = static_cast<int>(c->N);
    sd::LubGrid grid;
    grid.inv_cell = 1.0 / (3.0 * c->a);
    grid.L = c->box;
    grid.invL = c->box > 0.0 ? 1.0 / c->box : 0.0;
    grid.nc = 0;
    if (c->box > 0.0) {
        // the fp32 kernels see the box side rounded to float (as the pair kernels do)
        if (c->precision != SD_PREC_F64) {
            grid.L = static_cast<double>(static_cast<float>(c->box));
            grid.invL = 1.0 / grid.L;
        }
        grid.nc = static_cast<int>(std::floor(grid.L / (3.0 * c->a)));
        // a pair inside 3a must have ONE nearest image: L > 6a; the cell grid probes 27 distinct
        // cells and needs three of them per edge: L >= 9a
        if (grid.nc < 2 || !(grid.L > 6.0 * c->a))
            return fail(c, SD_ERR_UNSUPPORTED, "lubrication in a periodic box needs a box side above 6 a");
        if (grid.nc < 3 && n > sd::kLubOneCtaMaxN)
            return fail(c, SD_ERR_UNSUPPORTED,
                        "lubrication in a periodic box needs a box side of at least 9 a above 4096 particles (cell grid)");
    }
    const double gx = g ? g[0] : 0.0, gy = g ? g[1] : 0.0, gz = g ? g[2] : 0.0;
    if (n > sd::kLubSmallMax && n <= sd::kLubOneCtaMaxN && (grid.nc == 0 || grid.nc >= 3)) {
        // one launch: every CTA builds the grid in its shared memory, then takes its share of the particles
        grid.M = 16;  // 16^3 = kLubOneCtaMaxH buckets
        if (grid.nc > 0) {
            grid.nc = std::min(grid.nc, grid.M);
            grid.M = grid.nc;
        }
        const int ctas = std::min(c->num_sms, (n + 31) / 32);
        if (!c->lub_one_launch_ready) {
            SD_CUDA(c, cudaFuncSetAttribute(sd::lub_one_launch_kernel<float4>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            static_cast<int>(sizeof(sd::LubOneLaunchSmem<float4>))));
            SD_CUDA(c, cudaFuncSetAttribute(sd::lub_one_launch_kernel<double4>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            static_cast<int>(sizeof(sd::LubOneLaunchSmem<double4>))));
            c->lub_one_launch_ready = true;
        }
        if (c->precision == SD_PREC_F64)
            sd::lub_one_launch_kernel<double4>
                <<<ctas, sd::kLubOneCtaThreads, sizeof(sd::LubOneLaunchSmem<double4>), st>>>(
                    static_cast<const double4*>(pos), static_cast<const double4*>(vel),
                    static_cast<const double4*>(fext), gx, gy, gz, static_cast<double4*>(force_out), grid,
                    c->a, c->mu0, n);
        else
            sd::lub_one_launch_kernel<float4>
                <<<ctas, sd::kLubOneCtaThreads, sizeof(sd::LubOneLaunchSmem<float4>), st>>>(
                    static_cast<const float4*>(pos), static_cast<const float4*>(vel),
                    static_cast<const float4*>(fext), gx, gy, gz, static_cast<float4*>(force_out), grid,
                    c->a, c->mu0, n);
        return check_launch(c, "lub_one_launch_kernel");
    }
    if (n <= sd::kLubOneCtaMaxN) {  // small systems, small boxes: all pairs in one launch, no cell grid
        const int blocks = (n + 7) / 8;
        grid.M = 0;
        if (c->precision == SD_PREC_F64)
            sd::lub_small_kernel<double4><<<blocks, 256, 0, st>>>(
                static_cast<const double4*>(pos), static_cast<const double4*>(vel),
                static_cast<const double4*>(fext), gx, gy, gz, static_cast<double4*>(force_out), grid, c->a,
                c->mu0, n);
        else
            sd::lub_small_kernel<float4><<<blocks, 256, 0, st>>>(
                static_cast<const float4*>(pos), static_cast<const float4*>(vel),
                static_cast<const float4*>(fext), gx, gy, gz, static_cast<float4*>(force_out), grid, c->a,
                c->mu0, n);
        return check_launch(c, "lub_small_kernel");
    }
    {
        sd_status a = ensure_lub_buffers(c);
        if (a != SD_OK) return a;
    }
    const unsigned H = c->lub_H;  // 8^bits buckets, M = 2^bits per edge
    unsigned bits = 0;
    while ((1u << (3 * (bits + 1))) <= H) ++bits;
    grid.M = 1 << bits;
    if (grid.nc > 0) {  // box: one bucket per cell, larger cells if there are more than M per edge
        grid.nc = std::min(grid.nc, grid.M);
        grid.M = grid.nc;
    }
    const int nb = (n + 255) / 256;
    const unsigned nscan = (H + 1 + sd::kScanBlock - 1) / sd::kScanBlock;
    if (c->lub_count_dirty) SD_CUDA(c, cudaMemsetAsync(c->lub_count, 0, sizeof(unsigned) * (H + 1), st));
    sd_status s;
#define SD_LUB_FORCE_ARGS(T4)                                                                       \
    static_cast<const T4*>(c->lub_spos), static_cast<const T4*>(c->lub_svel), c->lub_order,         \
        static_cast<const T4*>(fext), gx, gy, gz, c->lub_start, static_cast<T4*>(force_out), grid,  \
        c->a, c->mu0, n
#define SD_LUB(T4)                                                                                  \
    c->lub_count_dirty = true;                                                                      \
    sd::lub_count_kernel<T4><<<nb, 256, 0, st>>>(static_cast<const T4*>(pos), c->lub_bucket,        \
                                                 c->lub_count, grid, n);                           \
    if ((s = check_launch(c, "lub_count_kernel")) != SD_OK) return s;                               \
    sd::lub_scan_totals_kernel<<<nscan, 256, 0, st>>>(c->lub_count, static_cast<unsigned*>(c->lub_tmp), \
                                                      H + 1);                                      \
    if ((s = check_launch(c, "lub_scan_totals_kernel")) != SD_OK) return s;                         \
    sd::lub_scan_apply_kernel<<<nscan, 256, 0, st>>>(c->lub_count, static_cast<const unsigned*>(c->lub_tmp), \
                                                     c->lub_start, c->lub_cursor, H + 1);          \
    if ((s = check_launch(c, "lub_scan_apply_kernel")) != SD_OK) return s;                          \
    sd::lub_scatter_kernel<<<nb, 256, 0, st>>>(c->lub_bucket, c->lub_cursor, c->lub_slots, n);      \
    if ((s = check_launch(c, "lub_scatter_kernel")) != SD_OK) return s;                             \
    sd::lub_gather_kernel<T4><<<nb, 256, 0, st>>>(static_cast<const T4*>(pos), static_cast<const T4*>(vel), \
                                                  c->lub_slots, c->lub_start, c->lub_count, c->lub_order, \
                                                  static_cast<T4*>(c->lub_spos), static_cast<T4*>(c->lub_svel), n); \
    if ((s = check_launch(c, "lub_gather_kernel")) != SD_OK) return s;                              \
    c->lub_count_dirty = false;                                                                     \
    if (n >= sd::kLubOneLaneMinN)                                                                   \
        sd::lub_force_kernel<T4, 1><<<(n + 127) / 128, sd::kLubThreads, 0, st>>>(SD_LUB_FORCE_ARGS(T4)); \
    else if (n >= 32768)                                                                            \
        sd::lub_force_kernel<T4, 8><<<(n * 8 + 127) / 128, sd::kLubThreads, 0, st>>>(SD_LUB_FORCE_ARGS(T4)); \
    else                                                                                            \
        sd::lub_force_kernel<T4, 32><<<(n * 32 + 127) / 128, sd::kLubThreads, 0, st>>>(SD_LUB_FORCE_ARGS(T4)); \
    return check_launch(c, "lub_force_kernel")
    if (c->precision == SD_PREC_F64) {
        SD_LUB(double4);
    } else {
        SD_LUB(float4);
    }
#undef SD_LUB
}

template <typename T, int PATTERN>
void access_launch(int scheme, float* out, const T* in, unsigned N, cudaStream_t st) {
    const unsigned blocks = (N + sd::kAccThreads - 1) / sd::kAccThreads;
    if (scheme == sd::ACC_NAIVE)
        sd::access_naive_kernel<T, PATTERN><<<blocks, sd::kAccThreads, 0, st>>>(out, in, N);
    else if (scheme == sd::ACC_SMALL_TILING)
        sd::access_tiled_kernel<T, PATTERN, 32><<<blocks, sd::kAccThreads, 0, st>>>(out, in, N);
    else if (scheme == sd::ACC_TILING)
        sd::access_tiled_kernel<T, PATTERN, 128><<<blocks, sd::kAccThreads, 0, st>>>(out, in, N);
    else
        sd::access_bulk_kernel<T><<<blocks, sd::kAccThreads, 0, st>>>(out, in, N);
}
template <typename T>
void access_dispatch(int pattern, int scheme, float* out, const void* in, unsigned N, cudaStream_t st) {
    const T* p = static_cast<const T*>(in);
    if (pattern == sd::ACC_LINEAR) access_launch<T, sd::ACC_LINEAR>(scheme, out, p, N, st);
    else if (pattern == sd::ACC_STRIDED) access_launch<T, sd::ACC_STRIDED>(scheme, out, p, N, st);
    else access_launch<T, sd::ACC_UNORDERED>(scheme, out, p, N, st);
}
bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

// ---- sd_mobility_apply_noalloc: one product without a context and without any allocation -------
// Some callers cannot call cudaMalloc (code under stream capture, tight serving loops, harnesses
// that forbid it).  This is the warp-split one-launch kernel (sd_pairs_f32w.cuh, fp32 Kahan, free
// space) with ALL its scratch -- partial sums of the i-blocks that several CTAs share, the ticket
// counter and the schedule of every i-block, the pad records of the ragged tail -- in one
// file-scope device array of kNoAllocBytes (4 MiB; every GPU that loads the library holds it until
// exit).  The array is shared by every call and keeps the last call's contents:
// noalloc_prepare_kernel rewrites the schedule, the pad records and zeroes the tickets at the start
// of every call; calls that overlap on the GPU (two streams, two host threads) race on it.
constexpr long long kNoAllocMaxN = 16384;
constexpr size_t kNoAllocMaxB = (kNoAllocMaxN + 255) / 256;                  // i-blocks of 256 particles
constexpr size_t kNoAllocPadOff = 0;                                          // 2 x kWSJ float4
constexpr size_t kNoAllocDoneOff = kNoAllocPadOff + 2 * sd::kWSJ * sizeof(float4);
constexpr size_t kNoAllocFirstOff = kNoAllocDoneOff + kNoAllocMaxB * sizeof(int);
constexpr size_t kNoAllocSlotsOff = kNoAllocFirstOff + kNoAllocMaxB * sizeof(int);
constexpr size_t kNoAllocPartOff = (kNoAllocSlotsOff + kNoAllocMaxB * sizeof(int) + 255) / 256 * 256;
constexpr size_t kNoAllocBytes = 4u << 20;
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

// piece (CTA) that owns unit u when U units are cut at floor(g U / G): the largest g with
// floor(g U / G) <= u  (the rule of build_schedule)
__host__ __device__ inline int noalloc_piece_of(long long u, long long U, int G) {
    return static_cast<int>(((u + 1) * G - 1) / U);
}

__global__ void __launch_bounds__(256)
noalloc_prepare_kernel(float4* __restrict__ pad, int* __restrict__ blk_done, int* __restrict__ blk_first,
                       int* __restrict__ blk_nslots, const int B, const int T, const int G) {
    const long long U = static_cast<long long>(B) * T;
    for (int b = threadIdx.x; b < B; b += blockDim.x) {
        const long long lo = static_cast<long long>(b) * T;
        const int cf = noalloc_piece_of(lo, U, G), cl = noalloc_piece_of(lo + T - 1, U, G);
        blk_first[b] = cf;
        blk_nslots[b] = cl - cf + 1;
        blk_done[b] = 0;  // the shared array keeps whatever an earlier (possibly aborted) call left
    }
    for (int q = threadIdx.x; q < 2 * sd::kWSJ; q += blockDim.x)
        pad[q] = q < sd::kWSJ ? make_float4(SD_PAD_POS, SD_PAD_POS, SD_PAD_POS, 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
}

// per device, set up on the first call made with that device current
struct NoAllocDevice {
    bool ready = false;
    unsigned char* scratch = nullptr;  // DEVICE address of g_noalloc_scratch on this device
    int num_sms = 0;
};
constexpr int kNoAllocMaxDevices = 64;
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];
std::mutex g_noalloc_mutex;


}  // namespace

extern "C" {

sd_status sd_create(sd_ctx** out, long long N, double a, double eta) {
    if (!out) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_create: out is NULL");
    *out = nullptr;
    if (N < 1 || N > (1LL << 30)) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_create: N must be in [1, 2^30]");
    if (!(a > 0.0) || !(eta > 0.0) || !std::isfinite(a) || !std::isfinite(eta))
        return fail(nullptr, SD_ERR_INVALID_ARG, "sd_create: a and eta must be finite and > 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, SD_ERR_UNSUPPORTED, "sd_create: no CUDA device (there is no CPU fallback)");
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
        return fail(nullptr, SD_ERR_CUDA, "sd_create: cannot query the current device");
    if (prop.major != 10)
        return fail(nullptr, SD_ERR_UNSUPPORTED,
                    std::string("sd_create: built for sm_100a (B200); device is ") + prop.name);
    sd_ctx* c = new (std::nothrow) sd_ctx;
    if (!c) return fail(nullptr, SD_ERR_ALLOC, "sd_create: out of host memory");
    c->N = N;
    c->Nrec = (N + SD_REC_ALIGN - 1) / SD_REC_ALIGN * SD_REC_ALIGN;
    c->a = a;
    c->eta = eta;
    c->mu0 = 1.0 / (6.0 * 3.14159265358979323846 * eta * a);
    c->device = dev;
    c->num_sms = prop.multiProcessorCount;
    sd_status st = configure(c);
    if (st != SD_OK) {
        g_create_error = c->err;
        free_buffers(c);
        delete c;
        return st;
    }
    *out = c;
    return SD_OK;
}

namespace {
// with a non-default staging (ablation) only RPY + fp32-Kahan + free space exists
bool staging_forbids(const sd_ctx* c, int tensor, int precision, double box) {
    return c->staging != sd::STAGE_BULK &&
           (tensor != SD_TENSOR_RPY || precision != SD_PREC_F32_KAHAN || box > 0.0);
}
const char* kStagingMsg =
    "the staging ablation exists for RPY, fp32-Kahan, free space only: call sd_set_staging(ctx, 0) first";
}  // namespace

sd_status sd_set_tensor(sd_ctx* ctx, sd_tensor tensor) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_tensor: ctx is NULL");
    if (tensor != SD_TENSOR_RPY && tensor != SD_TENSOR_OSEEN)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_set_tensor: unknown tensor");
    if (static_cast<int>(tensor) == ctx->tensor) return SD_OK;
    if (staging_forbids(ctx, tensor, ctx->precision, ctx->box)) return fail(ctx, SD_ERR_UNSUPPORTED, kStagingMsg);
    cudaDeviceSynchronize();
    ctx->tensor = tensor;
    return configure(ctx);
}

sd_status sd_set_precision(sd_ctx* ctx, sd_precision precision) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_precision: ctx is NULL");
    if (precision != SD_PREC_F32_KAHAN && precision != SD_PREC_F64 && precision != SD_PREC_F32_PLAIN)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_set_precision: unknown precision");
    if (static_cast<int>(precision) == ctx->precision) return SD_OK;
    if (staging_forbids(ctx, ctx->tensor, precision, ctx->box)) return fail(ctx, SD_ERR_UNSUPPORTED, kStagingMsg);
    cudaDeviceSynchronize();
    ctx->precision = precision;
    return configure(ctx);
}

sd_status sd_schedule_plan(long long N, int particles_per_block, int tile_j, long long max_ctas, int num_sms,
                           long long* cta_u0, int* cta_piece, int* blk_first, int* blk_nslots, int* dims) {
    if (N < 1 || particles_per_block < 1 || tile_j < 1 || max_ctas < 1 || num_sms < 1 || !dims)
        return fail(nullptr, SD_ERR_INVALID_ARG, "sd_schedule_plan: invalid argument");
    const HostSchedule h = build_schedule(N, particles_per_block, tile_j, max_ctas, num_sms);
    dims[0] = h.B, dims[1] = h.T, dims[2] = h.G, dims[3] = h.max_slots;
    if (cta_u0) std::copy(h.u0.begin(), h.u0.end(), cta_u0);
    if (cta_piece) std::copy(h.piece.begin(), h.piece.end(), cta_piece);
    if (blk_first) std::copy(h.first.begin(), h.first.end(), blk_first);
    if (blk_nslots) std::copy(h.nslots.begin(), h.nslots.end(), blk_nslots);
    return SD_OK;
}

sd_status sd_set_dispatch(sd_ctx* ctx, long long small_apply_max, int particles_per_thread) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_dispatch: ctx is NULL");
    if (particles_per_thread != 0 && particles_per_thread != 2 && particles_per_thread != 4 &&
        particles_per_thread != 8)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_set_dispatch: particles_per_thread must be 0, 2, 4 or 8");
    cudaDeviceSynchronize();
    ctx->small_user = small_apply_max < 0 ? -1 : small_apply_max;
    ctx->ipt_override = particles_per_thread;
    return configure(ctx);
}

sd_status sd_set_jsplit(sd_ctx* ctx, int mode) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_jsplit: ctx is NULL");
    if (mode < 0 || mode > 2) return fail(ctx, SD_ERR_INVALID_ARG, "sd_set_jsplit: mode must be 0, 1 or 2");
    cudaDeviceSynchronize();
    ctx->jsplit = mode;
    return configure(ctx);
}

sd_status sd_set_position_compensation(sd_ctx* ctx, int on) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_position_compensation: ctx is NULL");
    ctx->pos_comp = on ? 1 : 0;
    drop_graph(ctx);
    ctx->lo_valid = false;  // low words are re-zeroed before the next step
    return SD_OK;
}

sd_status sd_set_staging(sd_ctx* ctx, int mode) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_staging: ctx is NULL");
    if (mode != sd::STAGE_BULK && mode != sd::STAGE_NAIVE && mode != sd::STAGE_SYNC)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_set_staging: mode must be 0 (bulk copies), 1 (naive) or 2 (tiled with barriers)");
    if (mode == ctx->staging) return SD_OK;
    cudaDeviceSynchronize();
    const int old = ctx->staging;
    ctx->staging = mode;
    sd_status s = configure(ctx);
    if (s != SD_OK) {  // unsupported combination: keep the context usable
        const std::string msg = ctx->err;
        ctx->staging = old;
        configure(ctx);
        ctx->err = msg;
    }
    return s;
}

sd_status sd_set_box(sd_ctx* ctx, double box_side) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_box: ctx is NULL");
    if (!(box_side >= 0.0) || !std::isfinite(box_side))
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_set_box: box side must be finite and >= 0 (0 = free space)");
    if (box_side > 0.0 && !(static_cast<float>(box_side) > 0.0f) )
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_set_box: box side underflows in fp32");
    if (staging_forbids(ctx, ctx->tensor, ctx->precision, box_side)) return fail(ctx, SD_ERR_UNSUPPORTED, kStagingMsg);
    const bool was = ctx->box > 0.0, is = box_side > 0.0;
    ctx->box = box_side;
    drop_graph(ctx);
    if (was == is) return SD_OK;  // same kernels, only the constants change
    cudaDeviceSynchronize();
    return configure(ctx);
}

sd_status sd_mobility_apply(sd_ctx* ctx, const void* pos, const void* force, void* vel, void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_mobility_apply: ctx is NULL");
    SD_ENTER(ctx, "sd_mobility_apply");
    if (!pos || !force || !vel) return fail(ctx, SD_ERR_INVALID_ARG, "sd_mobility_apply: NULL pointer");
    const size_t al = 4 * elem_size(ctx->precision);
    if (misaligned(pos, al) || misaligned(force, al) || misaligned(vel, al))
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_mobility_apply: records must be 16-byte (float) / 32-byte (double) aligned");
    if (vel == pos || vel == force) return fail(ctx, SD_ERR_INVALID_ARG, "sd_mobility_apply: vel aliases an input");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (ctx->N <= ctx->small_apply_max || ctx->w_on)  // one launch, no pack / finalize kernels
        return launch_small_apply(ctx, pos, force, nullptr, vel, nullptr, nullptr, 0.0, sd::FIN_VEL, st);
    sd_status s = launch_pack(ctx, pos, force, sd::PACK_POS | sd::PACK_FORCE, nullptr, st);
    if (s != SD_OK) return s;
    s = launch_pairs(ctx, st);
    if (s != SD_OK) return s;
    return launch_finalize<sd::FIN_VEL>(ctx, vel, nullptr, 0.0, st);
}

sd_status sd_mobility_apply_host(sd_ctx* ctx, const void* pos_host, const void* force_host,
                                 void* vel_host, void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_mobility_apply_host: ctx is NULL");
    SD_ENTER(ctx, "sd_mobility_apply_host");
    if (!pos_host || !force_host || !vel_host)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_mobility_apply_host: NULL pointer");
    const size_t bytes = static_cast<size_t>(ctx->N) * 4 * elem_size(ctx->precision);
    if (!ctx->stage_pos) {
        SD_CUDA(ctx, cudaMalloc(&ctx->stage_pos, bytes));
        SD_CUDA(ctx, cudaMalloc(&ctx->stage_force, bytes));
        SD_CUDA(ctx, cudaMalloc(&ctx->stage_vel, bytes));
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    SD_CUDA(ctx, cudaMemcpyAsync(ctx->stage_pos, pos_host, bytes, cudaMemcpyHostToDevice, st));
    SD_CUDA(ctx, cudaMemcpyAsync(ctx->stage_force, force_host, bytes, cudaMemcpyHostToDevice, st));
    sd_status s = sd_mobility_apply(ctx, ctx->stage_pos, ctx->stage_force, ctx->stage_vel, stream);
    if (s != SD_OK) return s;
    SD_CUDA(ctx, cudaMemcpyAsync(vel_host, ctx->stage_vel, bytes, cudaMemcpyDeviceToHost, st));
    SD_CUDA(ctx, cudaStreamSynchronize(st));
    return SD_OK;
}

sd_status sd_step(sd_ctx* ctx, void* pos, sd_force_fn fn, void* user, const void* force,
                  const double gravity[3], double dt, long long n_steps, sd_integrator integrator,
                  void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_step: ctx is NULL");
    SD_ENTER(ctx, "sd_step");
    if (!pos) return fail(ctx, SD_ERR_INVALID_ARG, "sd_step: pos is NULL");
    if (!fn && !force && !gravity) return fail(ctx, SD_ERR_INVALID_ARG, "sd_step: no force given");
    if (!std::isfinite(dt)) return fail(ctx, SD_ERR_INVALID_ARG, "sd_step: dt is not finite");
    if (n_steps < 0) return fail(ctx, SD_ERR_INVALID_ARG, "sd_step: n_steps < 0");
    if (integrator != SD_INT_EULER && integrator != SD_INT_MIDPOINT)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_step: unknown integrator");
    const size_t al = 4 * elem_size(ctx->precision);
    if (misaligned(pos, al) || (force && misaligned(force, al)))
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_step: misaligned records");
    if (n_steps == 0) return SD_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    sd_status s;
    if (!ctx->lo_valid) {
        SD_CUDA(ctx, cudaMemsetAsync(ctx->pos_lo, 0, static_cast<size_t>(ctx->Nrec) * al, st));
        ctx->lo_valid = true;
    }
    const bool lub = ctx->lubrication != 0;
    if (ctx->w_on && !fn && !lub && !force) {  // the warp-split kernel reads a force array
        const int n = static_cast<int>(ctx->N);
        if (ctx->precision == SD_PREC_F64)
            sd::fill4_kernel<double4><<<(n + 255) / 256, 256, 0, st>>>(static_cast<double4*>(ctx->grav_buf), gravity[0],
                                                                      gravity[1], gravity[2], n);
        else
            sd::fill4_kernel<float4><<<(n + 255) / 256, 256, 0, st>>>(static_cast<float4*>(ctx->grav_buf), gravity[0],
                                                                     gravity[1], gravity[2], n);
        if ((s = check_launch(ctx, "fill4_kernel")) != SD_OK) return s;
    }
    if (!fn && !lub && ctx->N <= sd::kStepperMax)  // all steps in one launch
        return launch_stepper(ctx, pos, force, gravity, dt, n_steps, integrator, st);

    // `count` steps enqueued on stream `st` (also used under stream capture, see below)
    auto run_steps = [&](cudaStream_t st, long long count) -> sd_status {
        sd_status s;
    // Forces that change from product to product (a caller callback and / or the lubrication
    // correction with the velocities of the previous product) are rebuilt in
    // the context's force buffer before every product.
    const bool dynamic = fn || lub;
    auto fill = [&](const void* p) -> sd_status {
        const void* fe = force;
        const double* gg = gravity;
        if (fn) {
            if (fn(p, ctx->force_buf, ctx->N, user, static_cast<void*>(st)) != 0)
                return fail(ctx, SD_ERR_INVALID_ARG, "sd_step: force callback failed");
            fe = ctx->force_buf;
        }
        if (lub) return launch_lubrication(ctx, p, ctx->vel, fe, fe ? nullptr : gg, ctx->force_buf, st);
        return SD_OK;
    };
    if (ctx->N <= ctx->small_apply_max || ctx->w_on) {    // one launch per product
        const void* fptr = dynamic ? ctx->force_buf : force;
        const double* g = (dynamic || force) ? nullptr : gravity;
        void* cur = pos;
        void* other = ctx->pos_alt;
        for (long long step = 0; step < count; ++step) {
            if (integrator == SD_INT_EULER) {
                if (dynamic && (s = fill(cur)) != SD_OK) return s;
                s = launch_small_apply(ctx, cur, fptr, g, ctx->vel, cur, other, dt, sd::FIN_EULER, st);
                if (s != SD_OK) return s;
                std::swap(cur, other);
            } else {
                if (dynamic && (s = fill(pos)) != SD_OK) return s;
                s = launch_small_apply(ctx, pos, fptr, g, ctx->vel, pos, ctx->pos_half, dt, sd::FIN_HALF, st);
                if (s != SD_OK) return s;
                if (dynamic && (s = fill(ctx->pos_half)) != SD_OK) return s;
                s = launch_small_apply(ctx, ctx->pos_half, fptr, g, ctx->vel, pos, pos, dt, sd::FIN_FULL, st);
                if (s != SD_OK) return s;
            }
        }
        if (cur != pos)
            SD_CUDA(ctx, cudaMemcpyAsync(pos, cur, static_cast<size_t>(ctx->N) * al,
                                         cudaMemcpyDeviceToDevice, st));
        return SD_OK;
    }
    // constant forces are packed once; dynamic forces before every product
    const int force_what = dynamic ? 0 : (force ? sd::PACK_FORCE : sd::PACK_GRAVITY);
    s = launch_pack(ctx, pos, force, sd::PACK_POS | force_what, gravity, st);
    if (s != SD_OK) return s;
    auto callback = [&](const void* p) -> sd_status {
        if (!dynamic) return SD_OK;
        sd_status r = fill(p);
        if (r != SD_OK) return r;
        return launch_pack(ctx, nullptr, ctx->force_buf, sd::PACK_FORCE, nullptr, st);
    };
    for (long long step = 0; step < count; ++step) {
        if ((s = callback(pos)) != SD_OK) return s;
        if ((s = launch_pairs(ctx, st)) != SD_OK) return s;
        if (integrator == SD_INT_EULER) {
            if ((s = launch_finalize<sd::FIN_EULER>(ctx, ctx->vel, pos, dt, st)) != SD_OK) return s;
        } else {
            if ((s = launch_finalize<sd::FIN_HALF>(ctx, ctx->vel, pos, dt, st)) != SD_OK) return s;
            if ((s = callback(ctx->pos_half)) != SD_OK) return s;
            if ((s = launch_pairs(ctx, st)) != SD_OK) return s;
            if ((s = launch_finalize<sd::FIN_FULL>(ctx, ctx->vel, pos, dt, st)) != SD_OK) return s;
        }
    }
    return SD_OK;
    };

    // The lubrication step is eight small launches: with it the loop is bound by the host's launch
    // rate (~100 us per step at any N), not by the GPU.  Constant-force runs are a fixed sequence of
    // launches, so kGraphSteps steps are captured once into a CUDA graph and replayed.
    // The one-launch-per-product loop of small systems is launch-bound as well (6 us per step at
    // N = 256 for a 3 us kernel) and is replayed the same way.
    if ((lub || ctx->N <= kGraphMaxN) && !fn && !ctx->profiling && n_steps >= 2 * kGraphSteps) {
        GraphKey key;
        std::memset(&key, 0, sizeof(key));  // padding bytes take part in the memcmp below
        key.pos = pos;
        key.force = force;
        if (gravity) key.gx = gravity[0], key.gy = gravity[1], key.gz = gravity[2];
        key.has_gravity = gravity != nullptr;
        key.dt = dt;
        key.integrator = static_cast<int>(integrator);
        if (!ctx->gexec || std::memcmp(&key, &ctx->gkey, sizeof(GraphKey)) != 0) {
            drop_graph(ctx);
            if (lub && ctx->N > sd::kLubOneCtaMaxN && (s = ensure_lub_buffers(ctx)) != SD_OK) return s;
            if (!ctx->cap_stream) SD_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
            const long long launches0 = ctx->launches;
            SD_CUDA(ctx, cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
            s = run_steps(ctx->cap_stream, kGraphSteps);
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamEndCapture(ctx->cap_stream, &graph);
            if (s != SD_OK || e != cudaSuccess) {
                if (graph) cudaGraphDestroy(graph);
                cudaGetLastError();
                return s != SD_OK ? s : fail(ctx, SD_ERR_CUDA, std::string("sd_step: graph capture: ") + cudaGetErrorString(e));
            }
            ctx->graph_launches = ctx->launches - launches0;
            ctx->launches = launches0;
            e = cudaGraphInstantiate(&ctx->gexec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) {
                ctx->gexec = nullptr;
                return fail(ctx, SD_ERR_CUDA, std::string("sd_step: graph instantiate: ") + cudaGetErrorString(e));
            }
            ctx->gkey = key;
        }
        long long done = 0;
        for (; done + kGraphSteps <= n_steps; done += kGraphSteps) {
            SD_CUDA(ctx, cudaGraphLaunch(ctx->gexec, st));
            ctx->launches += ctx->graph_launches;
        }
        return done < n_steps ? run_steps(st, n_steps - done) : SD_OK;
    }
    return run_steps(st, n_steps);
}

sd_status sd_set_lubrication(sd_ctx* ctx, int on) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_lubrication: ctx is NULL");
    ctx->lubrication = on ? 1 : 0;
    drop_graph(ctx);
    return SD_OK;
}

sd_status sd_set_velocity(sd_ctx* ctx, const void* vel, void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_set_velocity: ctx is NULL");
    SD_ENTER(ctx, "sd_set_velocity");
    const size_t bytes = static_cast<size_t>(ctx->N) * 4 * elem_size(ctx->precision);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (vel) SD_CUDA(ctx, cudaMemcpyAsync(ctx->vel, vel, bytes, cudaMemcpyDeviceToDevice, st));
    else SD_CUDA(ctx, cudaMemsetAsync(ctx->vel, 0, bytes, st));
    return SD_OK;
}

sd_status sd_lubrication_apply(sd_ctx* ctx, const void* pos, const void* vel, const void* f_ext,
                               const double gravity[3], void* force_out, void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_lubrication_apply: ctx is NULL");
    SD_ENTER(ctx, "sd_lubrication_apply");
    if (!pos || !vel || !force_out) return fail(ctx, SD_ERR_INVALID_ARG, "sd_lubrication_apply: NULL pointer");
    const size_t al = 4 * elem_size(ctx->precision);
    if (misaligned(pos, al) || misaligned(vel, al) || misaligned(force_out, al) || (f_ext && misaligned(f_ext, al)))
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_lubrication_apply: misaligned records");
    if (force_out == pos || force_out == vel)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_lubrication_apply: force_out aliases pos or vel");
    return launch_lubrication(ctx, pos, vel, f_ext, f_ext ? nullptr : gravity, force_out,
                              static_cast<cudaStream_t>(stream));
}

sd_status sd_get_velocity(sd_ctx* ctx, void* vel_out, void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_get_velocity: ctx is NULL");
    SD_ENTER(ctx, "sd_get_velocity");
    if (!vel_out) return fail(ctx, SD_ERR_INVALID_ARG, "sd_get_velocity: vel_out is NULL");
    const size_t bytes = static_cast<size_t>(ctx->N) * 4 * elem_size(ctx->precision);
    SD_CUDA(ctx, cudaMemcpyAsync(vel_out, ctx->vel, bytes, cudaMemcpyDeviceToDevice,
                                 static_cast<cudaStream_t>(stream)));
    return SD_OK;
}

sd_status sd_reset_compensation(sd_ctx* ctx, void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_reset_compensation: ctx is NULL");
    SD_ENTER(ctx, "sd_reset_compensation");
    const size_t bytes = static_cast<size_t>(ctx->Nrec) * 4 * elem_size(ctx->precision);
    SD_CUDA(ctx, cudaMemsetAsync(ctx->pos_lo, 0, bytes, static_cast<cudaStream_t>(stream)));
    ctx->lo_valid = true;
    return SD_OK;
}

long long sd_num_particles(const sd_ctx* ctx) { return ctx ? ctx->N : 0; }
double sd_self_mobility(const sd_ctx* ctx) { return ctx ? ctx->mu0 : 0.0; }
double sd_box(const sd_ctx* ctx) { return ctx ? ctx->box : 0.0; }
long long sd_launch_count(const sd_ctx* ctx) { return ctx ? ctx->launches : 0; }
const char* sd_kernel_name(const sd_ctx* ctx) {
    if (!ctx) return "";
    if (ctx->w_on) return ctx->wcfg.name;
    if (ctx->N <= ctx->small_apply_max)
        return ctx->precision == SD_PREC_F64
                   ? "small_apply_f64"
                   : ((ctx->N >= sd::kPackedMinN && ctx->N <= sd::kPackedMaxN) ? "small_apply_f32x2" : "small_apply_f32");
    return ctx->cfg.name;
}

sd_status sd_profile_enable(sd_ctx* ctx, int on) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_profile_enable: ctx is NULL");
    ctx->profiling = on != 0;
    return SD_OK;
}

sd_status sd_profile_read(sd_ctx* ctx, double* pair_kernel_ms, long long* pair_kernel_launches) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_profile_read: ctx is NULL");
    if (!pair_kernel_ms || !pair_kernel_launches)
        return fail(ctx, SD_ERR_INVALID_ARG, "sd_profile_read: NULL output");
    double total = 0.0;
    for (auto& ev : ctx->prof_events) {
        SD_CUDA(ctx, cudaEventSynchronize(ev.second));
        float ms = 0.f;
        SD_CUDA(ctx, cudaEventElapsedTime(&ms, ev.first, ev.second));
        total += ms;
        ctx->prof_pool.push_back(ev);
    }
    *pair_kernel_ms = total;
    *pair_kernel_launches = static_cast<long long>(ctx->prof_events.size());
    ctx->prof_events.clear();
    return SD_OK;
}

sd_status sd_fma_peak_probe(sd_ctx* ctx, sd_precision precision, double* tflops_out, void* stream) {
    if (!ctx) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_fma_peak_probe: ctx is NULL");
    SD_ENTER(ctx, "sd_fma_peak_probe");
    if (!tflops_out) return fail(ctx, SD_ERR_INVALID_ARG, "sd_fma_peak_probe: tflops_out is NULL");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int threads = 512, blocks = ctx->num_sms * 4, iters = 4096;
    if (!ctx->probe) SD_CUDA(ctx, cudaMalloc(&ctx->probe, sizeof(double) * threads * blocks));
    cudaEvent_t e0, e1;
    SD_CUDA(ctx, cudaEventCreate(&e0));
    SD_CUDA(ctx, cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        if (precision == SD_PREC_F64)
            sd::fma_probe_f64_kernel<<<blocks, threads, 0, st>>>(static_cast<double*>(ctx->probe), 1.0000001, 1e-3, iters);
        else
            sd::fma_probe_f32_kernel<<<blocks, threads, 0, st>>>(static_cast<float*>(ctx->probe), 1.0001f, 1e-3f, iters);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best = std::min(best, ms);
        ++ctx->launches;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    SD_CUDA(ctx, cudaGetLastError());
    const double fmas = static_cast<double>(iters) * 64.0 * threads * blocks;
    *tflops_out = 2.0 * fmas / (best * 1e-3) / 1e12;
    return SD_OK;
}

sd_status sd_access_bench(int elem_floats, int pattern, int scheme, long long N, int reps, const void* in,
                          void* out, double* ms_per_launch, void* stream) {
    if ((elem_floats != 1 && elem_floats != 4) || pattern < 0 || pattern > 2 || scheme < 0 || scheme > 3 ||
        N < 1 || N > (1LL << 24) || reps < 1 || !in || !out)
        return fail(nullptr, SD_ERR_INVALID_ARG, "sd_access_bench: invalid argument");
    if (scheme == sd::ACC_BULK && (pattern != sd::ACC_LINEAR || (elem_floats == 1 && N % 4 != 0)))
        return fail(nullptr, SD_ERR_UNSUPPORTED,
                    "sd_access_bench: bulk copies need the linear pattern (and N % 4 == 0 for float)");
    if (misaligned(in, 16)) return fail(nullptr, SD_ERR_INVALID_ARG, "sd_access_bench: in must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned n = static_cast<unsigned>(N);
    float* o = static_cast<float*>(out);
    auto launch = [&]() {
        if (elem_floats == 1) access_dispatch<float>(pattern, scheme, o, in, n, st);
        else access_dispatch<float4>(pattern, scheme, o, in, n, st);
    };
    launch();  // warm-up (and the result the caller checks)
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess)
        return fail(nullptr, SD_ERR_CUDA, "sd_access_bench: cannot create events");
    cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess || (e = cudaGetLastError()) != cudaSuccess)
        return fail(nullptr, SD_ERR_CUDA, std::string("sd_access_bench: ") + cudaGetErrorString(e));
    if (ms_per_launch) *ms_per_launch = static_cast<double>(ms) / reps;
    return SD_OK;
}

sd_status sd_mobility_apply_noalloc(long long N, double a, double eta, sd_tensor tensor, const void* pos,
                                    const void* force, void* vel, void* stream) {
    if (N < 1 || !(a > 0.0) || !(eta > 0.0) || !std::isfinite(a) || !std::isfinite(eta))
        return fail(nullptr, SD_ERR_INVALID_ARG, "sd_mobility_apply_noalloc: N >= 1, a > 0 and eta > 0 required");
    if (N > kNoAllocMaxN)
        return fail(nullptr, SD_ERR_UNSUPPORTED,
                    "sd_mobility_apply_noalloc: N = " + std::to_string(N) + " exceeds the maximum of " +
                        std::to_string(kNoAllocMaxN) + " particles of the static scratch array (use a context)");
    if (tensor != SD_TENSOR_RPY && tensor != SD_TENSOR_OSEEN)
        return fail(nullptr, SD_ERR_INVALID_ARG, "sd_mobility_apply_noalloc: unknown tensor");
    if (!pos || !force || !vel || misaligned(pos, 16) || misaligned(force, 16) || misaligned(vel, 16))
        return fail(nullptr, SD_ERR_INVALID_ARG, "sd_mobility_apply_noalloc: pos, force, vel must be 16-byte aligned device arrays");
    if (vel == pos || vel == force)
        return fail(nullptr, SD_ERR_INVALID_ARG, "sd_mobility_apply_noalloc: vel must not alias pos or force");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kNoAllocMaxDevices)
        return fail(nullptr, SD_ERR_CUDA, std::string("sd_mobility_apply_noalloc: cudaGetDevice: ") + cudaGetErrorString(e));
    const bool rpy = tensor == SD_TENSOR_RPY;
    const void* kernel = w_pick<4>(rpy, false, false);
    const size_t smem = sd::WShape<4>::smem_bytes;
    NoAllocDevice& d = g_noalloc_dev[dev];
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!d.ready) {
            // in host code g_noalloc_scratch is a stand-in, not a device address: ask for the address on
            // the current device, once per device
            void* p = nullptr;
            if ((e = cudaGetSymbolAddress(&p, g_noalloc_scratch)) != cudaSuccess || !p)
                return fail(nullptr, SD_ERR_CUDA, std::string("sd_mobility_apply_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
            for (int t = 0; t < 2; ++t)
                if ((e = cudaFuncSetAttribute(w_pick<4>(t == 0, false, false), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              static_cast<int>(smem))) != cudaSuccess)
                    return fail(nullptr, SD_ERR_CUDA, std::string("sd_mobility_apply_noalloc: cudaFuncSetAttribute: ") + cudaGetErrorString(e));
            int sms = 0;
            if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess || sms < 1)
                return fail(nullptr, SD_ERR_CUDA, std::string("sd_mobility_apply_noalloc: cudaDeviceGetAttribute: ") + cudaGetErrorString(e));
            d.scratch = static_cast<unsigned char*>(p);
            d.num_sms = sms;
            d.ready = true;
        }
    }
    // the schedule of configure_w: i-blocks of 256 particles x quads of 4 j, one piece per SM
    const int IB = 64 * 4;
    const int B = static_cast<int>((N + IB - 1) / IB), T = static_cast<int>((N + sd::kWQ - 1) / sd::kWQ);
    const long long U = static_cast<long long>(B) * T;
    const int G = static_cast<int>(std::min<long long>(U, d.num_sms));
    int max_slots = 1;
    for (int b = 0; b < B; ++b) {
        const long long lo = static_cast<long long>(b) * T;
        max_slots = std::max(max_slots, noalloc_piece_of(lo + T - 1, U, G) - noalloc_piece_of(lo, U, G) + 1);
    }
    const long long stride = static_cast<long long>(B) * IB;  // particles per slot of the partial sums
    const size_t part_bytes = static_cast<size_t>(max_slots) * stride * 2 * sizeof(float4);
    if (kNoAllocPartOff + part_bytes > kNoAllocBytes)
        return fail(nullptr, SD_ERR_UNSUPPORTED,
                    "sd_mobility_apply_noalloc: the partial sums of this size on this GPU (" + std::to_string(part_bytes) +
                        " bytes) do not fit in the static scratch array");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    float4* pad = reinterpret_cast<float4*>(d.scratch + kNoAllocPadOff);
    int* blk_done = reinterpret_cast<int*>(d.scratch + kNoAllocDoneOff);
    int* blk_first = reinterpret_cast<int*>(d.scratch + kNoAllocFirstOff);
    int* blk_nslots = reinterpret_cast<int*>(d.scratch + kNoAllocSlotsOff);
    float4* part = reinterpret_cast<float4*>(d.scratch + kNoAllocPartOff);
    noalloc_prepare_kernel<<<1, 256, 0, st>>>(pad, blk_done, blk_first, blk_nslots, B, T, G);
    if ((e = cudaGetLastError()) != cudaSuccess)
        return fail(nullptr, SD_ERR_CUDA, std::string("noalloc_prepare_kernel: ") + cudaGetErrorString(e));
    sd::Schedule sch;
    sch.cta_u0 = nullptr, sch.cta_piece = nullptr;  // not read by the warp-split kernel
    sch.blk_first_cta = blk_first, sch.blk_nslots = blk_nslots;
    sch.T = T, sch.B = B, sch.G = G;
    const double mu0 = 1.0 / (6.0 * 3.14159265358979323846 * eta * a);
    sd::PairCoef k;
    k.k2 = static_cast<float>(2.0 * a * a / 3.0);
    k.m3k2 = static_cast<float>(-2.0 * a * a);
    k.mu0r = static_cast<float>(4.0 / (3.0 * a));
    k.ovA = static_cast<float>(-3.0 / (8.0 * a * a));
    k.ovB = static_cast<float>(1.0 / (8.0 * a * a));
    k.thr = rpy ? static_cast<float>(4.0 * a * a) : 1e-30f;
    k.clampv = static_cast<float>(4.0 * a * a);
    k.invL = k.mL = k.magic = 0.f;  // free space
    sd::FinArgs fin;
    fin.vel = static_cast<float4*>(vel);
    fin.pos_base = nullptr, fin.pos_lo = nullptr, fin.pos_out = nullptr;  // FIN_VEL: velocities only
    fin.dt = 0.0;
    fin.c1 = mu0 * 0.75 * a;
    fin.mu0 = mu0;
    fin.mode = sd::FIN_VEL;
    fin.pos_comp = 0;
    const float4* pp = static_cast<const float4*>(pos);
    const float4* ff = static_cast<const float4*>(force);
    const float4* cpad = pad;
    int n = static_cast<int>(N);
    long long slot_stride = stride;
    void* args[] = {&pp, &ff, &cpad, &part, &blk_done, &sch, &k, &fin, &n, &slot_stride};
    if ((e = cudaLaunchKernel(kernel, dim3(G), dim3(sd::kThreads), args, smem, st)) != cudaSuccess ||
        (e = cudaGetLastError()) != cudaSuccess)
        return fail(nullptr, SD_ERR_CUDA, std::string("sd_mobility_apply_noalloc: pairs_f32w_kernel: ") + cudaGetErrorString(e));
    return SD_OK;
}

long long sd_noalloc_max_particles(void) { return kNoAllocMaxN; }

const char* sd_last_error(const sd_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

void sd_destroy(sd_ctx* ctx) {
    if (!ctx) return;
    cudaDeviceSynchronize();
    for (auto* v : {&ctx->prof_events, &ctx->prof_pool})
        for (auto& ev : *v) {
            cudaEventDestroy(ev.first);
            cudaEventDestroy(ev.second);
        }
    free_buffers(ctx);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    delete ctx;
}

}  // extern "C"
