// api.cu -- C-ABI entry points of libbloch_b200 (include/bloch.h) and the per-block launch logic.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>

#include "internal.h"
#include "kernels.cuh"
#include "coils.cuh"
#include "coils_tc.cuh"
#include "coils_h.cuh"
#include "rf.cuh"
#include "seq.cuh"
#include "signal.cuh"

namespace bloch {
const char *last_error_cstr();
int collect_status(const bloch_plan *plan, int *flags_out);

namespace {

int cuda_fail(cudaError_t e, const char *what) {
    return fail(BLOCH_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define BLOCH_CUDA(call)                                         \
    do {                                                         \
        cudaError_t e_ = (call);                                 \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);      \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Per-device facts and one-time set-up, keyed by the CUDA device ordinal: SM count, compute capability, and whether
// the opt-in shared-memory limits of the kernels that need more than 48 KB have been raised ON THAT DEVICE
// (cudaFuncSetAttribute is per device, so a process that drives several GPUs sets it once on each).
constexpr int kMaxDevices = 64;
struct DeviceInfo {
    std::atomic<int> sms{0}, major{0};
    std::atomic<bool> seq_attr{false}, tc_attr{false}, h_attr{false};
};
DeviceInfo g_dev[kMaxDevices];

// the current device's slot, or nullptr when there is no usable device (host-only callers)
DeviceInfo *current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return nullptr;
    }
    if (dev < 0 || dev >= kMaxDevices) return nullptr;
    DeviceInfo *d = &g_dev[dev];
    if (d->sms.load(std::memory_order_acquire) == 0) {
        int sms = 0, major = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || sms <= 0) {
            (void)cudaGetLastError();
            return nullptr;
        }
        d->major.store(major, std::memory_order_relaxed);
        d->sms.store(sms, std::memory_order_release);
    }
    return d;
}

// ONE source for the SM count that sizes launch shapes: workspace sizing and workspace carving both use it, so they
// cannot disagree; 148 (a B200) when no device is present, which keeps bloch_plan_workspace_bytes a host function.
int sm_count_cached() {
    const DeviceInfo *d = current_device();
    return d ? d->sms.load(std::memory_order_relaxed) : 148;
}

int check_arch() {
    const DeviceInfo *d = current_device();
    if (!d) return fail(BLOCH_ECUDA, "no usable CUDA device is current");
    if (d->major.load(std::memory_order_relaxed) != 10)
        return fail(BLOCH_EARCH, "device is not compute capability 10.x (built for sm_100a only)");
    return BLOCH_OK;
}

// Signal-kernel launch shape for a block with n_pts evaluated points.
struct SigShape {
    int P;
    int ptiles;
    int chunks;
    int spins_per_chunk;
    int threads;  // CTA size: kSigThreads, or fewer for blocks of fewer samples (every thread owns a sample)
};

// max_P: 8, or 4 for fp64-phase motion plans (P = 8 would need 172 registers there: config 3m 2.09 -> 2.47 ms)
SigShape sig_shape(const bloch_plan *plan, int64_t n_pts, int64_t n_spins, int sm_count, int max_P) {
    SigShape s;
    const int forceP = plan->opt[BLOCH_OPT_SIGNAL_P];
    // 8 adjacent samples per thread when the block is long enough (config 4: 42.5 -> 35.6 ms together with the
    // geometric decay; ~100 registers, 2 CTAs per SM), else 4 / 2 / 1
    s.P = forceP ? forceP : (n_pts >= 8 * kSigThreads && max_P >= 8 ? 8 : (n_pts >= 4 * kSigThreads ? 4 : (n_pts >= 2 * kSigThreads ? 2 : 1)));
    if (s.P != 1 && s.P != 2 && s.P != 4 && s.P != 8) s.P = 1;
    // a readout of fewer than 256 samples (Cartesian lines) gets CTAs of just enough warps and more of them per SM,
    // so that the spins are split over all lanes instead of leaving 256 - n_pts threads of every CTA idle
    s.threads = kSigThreads;
    if (s.P == 1 && n_pts < kSigThreads && !plan->opt[BLOCH_OPT_SIGNAL_FIXED_CTA])
        s.threads = (int)std::max<int64_t>(32, (n_pts + 31) / 32 * 32);
    s.ptiles = (int)((n_pts + (int64_t)s.threads * s.P - 1) / ((int64_t)s.threads * s.P));
    const int per_sm = std::min(plan->opt[BLOCH_OPT_SIGNAL_CTAS_PER_SM] * (kSigThreads / s.threads), 12);
    const int64_t target = (int64_t)sm_count * per_sm;
    int64_t chunks = (target + s.ptiles - 1) / s.ptiles;
    const int64_t max_chunks = (n_spins + 31) / 32;
    if (chunks > max_chunks) chunks = max_chunks;
    if (chunks < 1) chunks = 1;
    if (chunks > 65535) chunks = 65535;
    s.spins_per_chunk = (int)std::max<int64_t>(1, (n_spins + chunks - 1) / chunks);
    s.chunks = (int)std::max<int64_t>(1, (n_spins + s.spins_per_chunk - 1) / s.spins_per_chunk);
    return s;
}

int sig_max_P(const bloch_plan *plan) {
    return (plan->info.phase_mode == BLOCH_PHASE_FP64 && plan->info.motion_mode != BLOCH_MOTION_NONE) ? 4 : 8;
}

// Launch shape of a precession block: blocks that go to signal_lin_kernel (Block::lin_pts) are chunked as P = 8 blocks
// whatever the plan (their kernel holds 2 CTAs per SM also with fp64 phase and motion).
SigShape block_shape(const bloch_plan *plan, const Block &b, int64_t n_spins, int sm_count) {
    const bool lin = b.lin_pts > 0 && plan->opt[BLOCH_OPT_SIGNAL_LIN];
    if (!lin) return sig_shape(plan, b.adc_count, n_spins, sm_count, sig_max_P(plan));
    // signal_lin_kernel: one thread per group of kLinP samples, 2 CTAs of 256 threads per SM (or proportionally more
    // CTAs of fewer warps for short blocks), the spins split over enough chunks to fill the machine
    SigShape s;
    s.P = kLinP;
    const int64_t n_groups = b.lin_pts / kLinP;
    s.threads = (int)std::min<int64_t>(kSigThreads, (n_groups + 31) / 32 * 32);
    s.ptiles = (int)((n_groups + s.threads - 1) / s.threads);
    const int per_sm = std::min(2 * (kSigThreads / s.threads), 8);
    int64_t chunks = ((int64_t)sm_count * per_sm + s.ptiles - 1) / s.ptiles;
    chunks = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(chunks, (n_spins + 31) / 32), 65535));
    s.spins_per_chunk = (int)std::max<int64_t>(1, (n_spins + chunks - 1) / chunks);
    s.chunks = (int)std::max<int64_t>(1, (n_spins + s.spins_per_chunk - 1) / s.spins_per_chunk);
    return s;
}

// Partial-sum buffer (a7): consecutive ADC-bearing precession blocks with the same launch shape share one
// buffer P[chunk][points of the batch] and ONE second-pass launch, up to kPartialCapBytes; at least the
// largest single block always fits.
constexpr size_t kPartialCapBytes = size_t(512) << 20;

size_t partial_elems_for(const bloch_plan *plan, int64_t n_spins, int sm_count) {
    size_t worst = 1, total = 0;
    for (const Block &b : plan->blocks) {
        if (b.type != kBlockPrecession || b.adc_count == 0) continue;
        const SigShape s = block_shape(plan, b, n_spins, sm_count);
        const size_t e = size_t(s.chunks) * size_t(b.adc_count);
        worst = std::max(worst, e);
        total += e;
    }
    return std::max(worst, std::min(total, kPartialCapBytes / sizeof(float2)));
}

// Launch shape of the whole-sequence kernel (seq.cuh): one CTA per chunk of spins, chunk = spins per SM rounded
// up to whole warps; ok = the plan and n_spins qualify, use = bloch_simulate takes it (plan->path, heuristic).
struct SeqShape {
    bool ok, use;
    int n_ctas, chunk, rf_warps, sig_warps, threads, min_items;
    int ring_slots, slot_stride;  // partial-row ring: [ring_slots][n_ctas][slot_stride] float2 ([..][n_ctas][nc][slot_stride] with coils)
    int nc;                       // weights per spin record with receive coils (4 or 8), else 0
    SeqRoles roles;
    size_t smem, partial_elems, ticket_off;  // float2 elements of the partial area; where the tickets start in it
};
// The ring holds the partial rows of the kSeqRingSlots blocks between "written" and "summed over CTAs" (seq.cuh), so
// its size is set by the LARGEST block, not by the sequence (config 5: 8 x 147 x 1024 x 8 B = 9.6 MB, where one row per
// CTA over the whole sequence was 1.2 GB); the path is unavailable only if that passes kSeqRingCapBytes (a single block
// of > 900k samples on 148 SMs; max_block_points cuts such blocks).
constexpr size_t kSeqRingCapBytes = size_t(8) << 30;

// L2-resident partial rows: with coils a slot is nc times larger, so fewer slots are kept once the ring passes this
constexpr size_t kSeqRingL2Bytes = size_t(48) << 20;

SeqShape seq_shape(const bloch_plan *plan, int64_t n_spins, int sm_count, int n_coils = 0) {
    SeqShape q{};
    const bloch_plan_info &inf = plan->info;
    // receive coils: up to 8 in the one launch, SUM_ALL plans; more take the per-block kernels
    if (n_coils < 0 || n_coils > 8 || (n_coils > 0 && inf.output_mode != BLOCH_OUT_SUM_ALL)) return q;
    q.nc = n_coils == 0 ? 0 : (n_coils <= 4 ? 4 : 8);
    // PER_SPIN plans qualify when every block holds only a few samples (dictionary mode: the RF thread that owns
    // the spin evaluates them itself, no signal warps)
    const bool ps = inf.output_mode == BLOCH_OUT_PER_SPIN;
    if ((inf.output_mode != BLOCH_OUT_SUM_ALL && !(ps && inf.max_block_adc <= 16)) ||
        inf.motion_mode != BLOCH_MOTION_NONE || inf.phase_mode != BLOCH_PHASE_FP32 || n_spins <= 0 ||
        plan->path == BLOCH_PATH_PER_BLOCK)
        return q;
    const int64_t per_sm = (n_spins + sm_count - 1) / sm_count;
    q.chunk = (int)std::max<int64_t>(32, (per_sm + 31) / 32 * 32);
    q.rf_warps = q.chunk / 32;
    // Roles per warp.  A warp runs on SM sub-partition (warp id mod 4); the RF warps are spread as evenly as they go
    // (the producer's sub-partition 0 takes an extra one last) and every sub-partition gets sig_base signal warps plus
    // sig_extra for every RF warp it holds fewer than the fullest one, so that all four carry about the same load.
    // Measured on config 5 (14 RF warps: 3,4,4,3): signal warps 3,1,1,3 124.1 ms; 3,2,2,3 125.9; 2,1,1,2 128.4;
    // 1,1,1,1 144.8; 2,2,2,2 133.6; 5,1,1,5 127.0.  With the 31-instruction RF step (rf.cuh, tier -1) the RF warps
    // got faster and the balance moved: 3,1,1,3 124.2 ms, 4,2,2,4 119.3, 3,2,2,3 119.8, 4,1,1,4 122.7, 3,3,3,3 121.6;
    // config 2 (4 RF warps, 16 RF steps per ADC sample) is indifferent (1,1,1,1 2.108 ms, 2,2,2,2 2.128).  Default: two
    // extra per missing RF warp, and a base that brings the total to about 0.85 signal warps per RF warp at one ADC
    // sample per RF step, scaled by the sequence's samples per RF step within [0.5, 1.25].
    int rf_per[4], sig_per[4], cnt_per[4];
    for (int k = 0; k < 4; ++k) rf_per[k] = q.rf_warps / 4;
    { const int order[4] = {1, 2, 3, 0}; for (int e = 0; e < q.rf_warps % 4; ++e) ++rf_per[order[e]]; }
    const int rf_max = *std::max_element(rf_per, rf_per + 4);
    // -1: two per missing RF warp; none with coils, where the signal warps are the heavier load and an equal number per
    // sub-partition is the better balance (config 5 x 4 coils: 4,4,4,4 162.6 ms against 168.8 for 5,3,3,5; x 8 coils
    // 205.2 against 213.0)
    const int sig_extra = plan->opt[BLOCH_OPT_SEQ_SIG_EXTRA] < 0 ? (q.nc > 0 ? 0 : 2)
                                                                 : std::min(plan->opt[BLOCH_OPT_SEQ_SIG_EXTRA], 7);
    int deficit = 0;
    for (int k = 0; k < 4; ++k) deficit += rf_max - rf_per[k];
    // with coils an evaluation costs (15 + 4 nc) / 15 of a plain one and has no P > 1 savings: ask for as many signal
    // warps as fit (the loop below gives warps back until the CTA holds 1024 threads)
    const double adc_per_rf = (inf.n_rf_steps > 0 ? double(inf.n_adc) / double(inf.n_rf_steps) : 1.0) *
                              (q.nc > 0 ? (19.0 + 4.0 * q.nc) / 15.0 : 1.0);
    const double adc_cap = q.nc > 0 ? 4.0 : 1.25;
    const int target = std::max(4, (int)std::lround(0.85 * q.rf_warps * std::min(std::max(adc_per_rf, 0.5), adc_cap)));
    const int auto_base = std::max(1, (target - sig_extra * deficit + 2) / 4);
    const int sig_base = plan->opt[BLOCH_OPT_SEQ_SIG_BASE] < 0 ? std::min(auto_base, 7)
                                                               : std::min(plan->opt[BLOCH_OPT_SEQ_SIG_BASE], 7);
    auto total_warps = [&](int base, int extra) {
        int top = 0;
        for (int k = 0; k < 4; ++k) {
            sig_per[k] = ps ? 0 : base + extra * (rf_max - rf_per[k]);
            cnt_per[k] = rf_per[k] + sig_per[k] + (k == 0 ? 1 : 0);
            if (cnt_per[k] > 0) top = std::max(top, (cnt_per[k] - 1) * 4 + k + 1);
        }
        return top;
    };
    int base = sig_base, extra = sig_extra;
    while (total_warps(base, extra) > kSeqMaxThreads / 32 && (extra > 0 || base > 0)) {
        if (base > 2) --base;          // give up base warps down to two per sub-partition first,
        else if (extra > 0) --extra;   // then the balancing extras,
        else --base;                   // then the rest
    }
    const int n_warps = total_warps(base, extra);
    // AUTO wants the whole set of signal warps, or at least two per sub-partition next to the balancing extras
    // (20 RF warps: 18.1 ms with 2 per sub-partition against 19.2 per-block and 21.4 with 1)
    const bool full_layout = (base == sig_base || base >= 2) && extra == sig_extra;
    q.sig_warps = sig_per[0] + sig_per[1] + sig_per[2] + sig_per[3];
    if (n_warps > kSeqMaxThreads / 32 || (!ps && q.sig_warps < 1))
        return q;  // no room beside the RF warps: more than 29 x 32 spins per SM (31 x 32 for PER_SPIN)
    {
        int rf_next = 0;
        for (int w = 0; w < kSeqMaxThreads / 32; ++w) q.roles.role[w] = (signed char)kRoleIdle;
        for (int k = 0; k < 4; ++k) {
            int slot = k;
            if (k == 0) { q.roles.role[slot] = (signed char)kRoleProducer; slot += 4; }
            for (int r = 0; r < rf_per[k]; ++r, slot += 4) q.roles.role[slot] = (signed char)0;  // index set below
            for (int g = 0; g < sig_per[k]; ++g, slot += 4) q.roles.role[slot] = (signed char)kRoleSignal;
        }
        for (int w = 0; w < n_warps; ++w)
            if (q.roles.role[w] == 0) q.roles.role[w] = (signed char)rf_next++;
        q.roles.n_sig_warps = q.sig_warps;
    }
    q.threads = 32 * n_warps;
    q.min_items = std::max(1, q.sig_warps * plan->opt[BLOCH_OPT_SEQ_ITEMS_X4] / 4);  // 0: always the largest P (config 5: 127.6 ms against 131.1 with one item per warp)
    q.n_ctas = (int)((n_spins + q.chunk - 1) / q.chunk);
    q.smem = seq_smem_bytes(q.chunk, q.nc);
    if (q.smem > size_t(227) * 1024) return q;
    if (inf.max_block_adc > INT32_MAX / 2) return q;
    q.slot_stride = (int)std::max<int64_t>(32, (inf.max_block_adc + 31) / 32 * 32);
    q.ring_slots = kSeqRingSlots;
    if (ps) { q.ring_slots = 1; q.slot_stride = 32; }  // PER_SPIN: no partial rows at all
    const size_t slot_elems = size_t(q.n_ctas) * size_t(std::max(q.nc, 1)) * size_t(q.slot_stride);
    // coils: keep the ring in L2 if that leaves at least lag + 2 slots (the CTAs may then drift 2 blocks apart)
    while (q.nc > 0 && q.ring_slots > kSeqReduceLag + 2 && size_t(q.ring_slots) * slot_elems * sizeof(float2) > kSeqRingL2Bytes)
        --q.ring_slots;
    const size_t ring_elems = ps ? 0 : size_t(q.ring_slots) * slot_elems;
    if (ring_elems * sizeof(float2) > kSeqRingCapBytes) return q;
    q.ticket_off = (ring_elems + 31) / 32 * 32;
    q.partial_elems = q.ticket_off + (size_t(2) * size_t(std::max<int64_t>(plan->n_adc_blocks, 1)) * sizeof(int) + 7) / 8;
    q.ok = true;
    // AUTO: the fused kernel pays when the excitation is a fair share of the work and the full set of signal warps
    // fits beside the RF warps (its readout runs on sig_warps warps per SM only).  Measured, fused / per-block ms:
    // N_rf/N_adc = 0.98: 13.1 / 15.5 at 65,536 spins, 42.1 / 29.4 at 131,044 (3 signal warps left);
    // 0.49: 5.97 / 6.17 at 65,536, 22.2 / 11.3 at 131,072;  0.06: 1.05 / 0.84 at 65,522.
    q.use = plan->path == BLOCH_PATH_FUSED || (4 * inf.n_rf_steps >= inf.n_adc && (ps || full_layout));
    // Coils under AUTO: the 8-wide sums cost ~50 issue slots per evaluation on the FMA pipe, so once a block holds
    // enough (spin, sample) pairs to fill the tcgen05 kernel the per-block launches win.  Measured, fused / per-block
    // ms: config 5 x 8 coils (6.7e7 pairs per block) 205.2 / 186.6; config 2 x 8 coils (1.0e6) 2.22 / 3.36; up to 4
    // coils the launch wins on both (config 5 x 4: 162.6 / 206.8; config 2 x 4: 2.13 / 3.19).
    if (q.nc == 8 && plan->path != BLOCH_PATH_FUSED && plan->opt[BLOCH_OPT_COIL_TC] != 0 &&
        n_spins * inf.max_block_adc >= (int64_t(1) << 24))
        q.use = false;
    return q;
}

// Multi-coil signal kernel (coils.cuh): P = 2 adjacent samples per thread (8 x P accumulators), grid as sig_shape.
// tc: the tcgen05 kernel (coils_tc.cuh): 128 samples per CTA of 288 threads, 2 CTAs per SM, chunks of whole 16-spin stages
bool coil_use_tc(const bloch_plan *plan, int64_t n_spins, int n_coils) {
    // BLOCH_OPT_COIL_TC: 0 = never; otherwise whenever it applies: fp32 phase, static spins (moving spins and fp64 phase:
    // the FFMA kernel) and
    //   1 (3xTF32 kernel, coils_tc.cuh): more than 4 coils -- one pass costs the same for 8, 16 and 32 coils (config 4:
    //     93-107 ms) and beats the FFMA kernel from its first pass of 8 (121 ms); up to 4 coils the 4-wide FFMA kernel
    //     (93 ms) stays;
    //   -1 (default) / 2 (FP16 kernel, coils_h.cuh): any number of coils once there are 4096 spins -- a pass of up to 8
    //     coils takes 76.9 ms on config 4, less than the 4-wide FFMA kernel's 93.2 for 1 to 4 coils.
    const int mode = plan->opt[BLOCH_OPT_COIL_TC];
    if (mode == 0 || n_coils < 1 || plan->info.phase_mode != BLOCH_PHASE_FP32 || plan->info.motion_mode != BLOCH_MOTION_NONE)
        return false;
    return n_coils > 4 || (mode != 1 && n_spins >= 4096);
}

// Multi-coil receive inside the whole-sequence kernel (seq_kernel<false, NC>): when the plan takes that path for
// n_spins and there are at most 8 coils.  Everything that sizes or carves the workspace asks this ONE function.
bool coil_use_fused(const bloch_plan *plan, int64_t n_spins, int sm_count, int n_coils) {
    if (n_coils <= 0) return false;
    const SeqShape q = seq_shape(plan, n_spins, sm_count, n_coils);
    return q.ok && q.use;
}

// which tensor-core kernel: FP16 operands (coils_h.cuh, 2 instructions per 8 spins) or 3xTF32 (coils_tc.cuh, 4)
// Measured on config 4 (signal kernels, per simulation): 8 coils 93.2 -> 76.9 ms, 16 coils 94.2 -> 74.1, 32 coils
// 106.4 -> 71.3; rounded (not truncated) operand pieces: errors against the oracle 2-3x smaller.  -1 (default) and 2:
// FP16; 1: 3xTF32.
bool coil_tc_fp16(const bloch_plan *plan) { return plan->opt[BLOCH_OPT_COIL_TC] != 1; }

SigShape coil_shape(int64_t n_pts, int64_t n_spins, int sm_count, int ncp, bool tc) {
    if (tc) {
        SigShape s;
        s.P = 1;
        s.threads = 256;
        s.ptiles = (int)((n_pts + kTcM - 1) / kTcM);
        int64_t chunks = std::max<int64_t>(1, ((int64_t)sm_count * 2) / s.ptiles);  // one wave of 2 CTAs per SM
        chunks = std::min<int64_t>(chunks, std::max<int64_t>(1, (n_spins + 255) / 256));
        chunks = std::min<int64_t>(chunks, 65535);
        const int64_t per = (n_spins + chunks - 1) / chunks;
        s.spins_per_chunk = (int)std::max<int64_t>(kTcStageSpins, (per + kTcStageSpins - 1) / kTcStageSpins * kTcStageSpins);
        s.chunks = (int)std::max<int64_t>(1, (n_spins + s.spins_per_chunk - 1) / s.spins_per_chunk);
        return s;
    }
    SigShape s;
    s.P = n_pts >= 2 * kSigThreads ? 2 : 1;
    s.threads = n_pts < kSigThreads ? (int)std::max<int64_t>(32, (n_pts + 31) / 32 * 32) : kSigThreads;  // as sig_shape
    s.ptiles = (int)((n_pts + (int64_t)s.threads * s.P - 1) / ((int64_t)s.threads * s.P));
    const int per_sm = std::min((ncp == 8 ? 2 : 4) * (kSigThreads / s.threads), 12);  // resident CTAs per SM (96 / 64 registers)
    int64_t chunks = ((int64_t)sm_count * per_sm + s.ptiles - 1) / s.ptiles;
    chunks = std::min<int64_t>(std::max<int64_t>(chunks, 1), std::min<int64_t>((n_spins + 31) / 32, 65535));
    chunks = std::max<int64_t>(chunks, 1);
    s.spins_per_chunk = (int)std::max<int64_t>(1, (n_spins + chunks - 1) / chunks);
    s.chunks = (int)std::max<int64_t>(1, (n_spins + s.spins_per_chunk - 1) / s.spins_per_chunk);
    return s;
}

size_t coil_partial_elems_for(const bloch_plan *plan, int64_t n_spins, int sm_count, int ncp, bool tc) {
    size_t worst = 1;
    for (const Block &b : plan->blocks) {
        if (b.type != kBlockPrecession || b.adc_count == 0) continue;
        const SigShape s = coil_shape(b.adc_count, n_spins, sm_count, ncp, tc);
        worst = std::max(worst, size_t(ncp) * size_t(s.chunks) * size_t(b.adc_count));
    }
    return worst;
}

// rows of the signal buffer: 1 (SUM_ALL), n_spins (PER_SPIN), n_spins / group_size (GROUPED)
size_t signal_rows(const bloch_plan *plan, int64_t n_spins) {
    if (plan->info.output_mode == BLOCH_OUT_PER_SPIN) return size_t(n_spins);
    if (plan->info.output_mode == BLOCH_OUT_GROUPED) return size_t(n_spins) / size_t(std::max(1, plan->info.group_size));
    return 1;
}

struct Workspace {
    float4 *A, *C, *S;
    double4 *Ad;     // fp64-phase plans only
    float4 *V;       // motion plans only: (vx, vy, vz, 0)
    double4 *Vd;     // motion + fp64 phase
    unsigned *scal;  // device scalars: [0] = max 1/T2 (float bits)
    float2 *partial;
    size_t partial_elems;
    float2 *W;       // multi-coil receive only: weights repacked as [pass][spin][4]
    float4 *Sp;      // FP16 tensor-core coil kernel only: block-start states in polar form
    size_t bytes;
};

// Layout of the caller's workspace.  sm_count = 148 is used for sizing when no device is present so that
// bloch_plan_workspace_bytes is a pure host function.
Workspace carve(const bloch_plan *plan, int64_t n_spins, void *base, int sm_count, int n_coils = 0) {
    Workspace w{};
    w.partial_elems = 0;
    size_t off = 0;
    auto take = [&](size_t bytes) {
        void *p = base ? (void *)((unsigned char *)base + off) : nullptr;
        off = align_up(off + bytes, kAlign);
        return p;
    };
    w.A = (float4 *)take(size_t(n_spins) * sizeof(float4));
    w.C = (float4 *)take(size_t(n_spins) * sizeof(float4));
    w.S = (float4 *)take(size_t(n_spins) * sizeof(float4));
    w.Ad = plan->info.phase_mode == BLOCH_PHASE_FP64 ? (double4 *)take(size_t(n_spins) * sizeof(double4)) : nullptr;
    const bool mo = plan->info.motion_mode != BLOCH_MOTION_NONE;
    w.V = mo ? (float4 *)take(size_t(n_spins) * sizeof(float4)) : nullptr;
    w.Vd = (mo && plan->info.phase_mode == BLOCH_PHASE_FP64) ? (double4 *)take(size_t(n_spins) * sizeof(double4)) : nullptr;
    w.scal = (unsigned *)take(kAlign);
    size_t pbytes = kAlign;
    if (plan->info.output_mode == BLOCH_OUT_SUM_ALL) {
        const SeqShape q = seq_shape(plan, n_spins, sm_count, n_coils);
        if (n_coils > 0 && !(q.ok && q.use)) {
            const bool tc_ = coil_use_tc(plan, n_spins, n_coils);
            w.partial_elems = coil_partial_elems_for(plan, n_spins, sm_count, tc_ ? tc_coils_per_pass(n_coils) : coils_per_pass(n_coils), tc_);
        }
        else w.partial_elems = (q.ok && q.use) ? q.partial_elems : partial_elems_for(plan, n_spins, sm_count);
        pbytes = w.partial_elems * sizeof(float2);
    }
    w.partial = (float2 *)take(pbytes);
    const bool tc_ws = n_coils > 0 && coil_use_tc(plan, n_spins, n_coils) && !coil_use_fused(plan, n_spins, sm_count, n_coils);
    const int ncp = tc_ws ? tc_coils_per_pass(n_coils) : coils_per_pass(n_coils);
    const size_t n_pass = size_t((n_coils + ncp - 1) / ncp);
    // the tcgen05 kernel takes its weights as ready-made B tiles: 2048 B per 8 spins (spins padded to whole stages)
    const size_t n_pad = (size_t(n_spins) + kTcStageSpins - 1) / kTcStageSpins * kTcStageSpins;
    const size_t w_bytes = tc_ws ? n_pass * (n_pad / 8) * tc_bgroup(ncp)
                                                                       : n_pass * size_t(n_spins) * ncp * sizeof(float2);
    w.W = n_coils > 0 ? (float2 *)take(w_bytes) : nullptr;
    w.Sp = (tc_ws && coil_tc_fp16(plan)) ? (float4 *)take(size_t(n_spins) * sizeof(float4)) : nullptr;
    w.bytes = off;
    return w;
}

struct Taps {
    const bloch_plan *plan;
    cudaStream_t stream;
    size_t used = 0;
    int mark(int kind) {
        if (!plan->profiling) return BLOCH_OK;
        if (used == plan->events.size()) {
            cudaEvent_t e;
            BLOCH_CUDA(cudaEventCreate(&e));
            plan->events.push_back((void *)e);
        }
        BLOCH_CUDA(cudaEventRecord((cudaEvent_t)plan->events[used], stream));
        if (plan->event_kind.size() <= used) plan->event_kind.resize(used + 1);
        plan->event_kind[used] = kind;
        ++used;
        return BLOCH_OK;
    }
};

// remember the largest launch of a kind (threads in flight) for bloch_plan_last_kernel
void note_kernel(const bloch_plan *plan, int kind, int64_t grid, int block, const char *fmt, int a = 0, int b = 0, int c = 0,
                 int d = 0) {
    KernelNote &k = plan->last_kernel[kind];
    if (grid * block < k.grid * k.block) return;
    std::snprintf(k.name, sizeof k.name, fmt, a, b, c, d);
    k.grid = grid;
    k.block = block;
}

}  // namespace

// Evaluates and clears the findings pack_kernel left in plan->h_status (see bloch_plan_status in bloch.h).
int collect_status(const bloch_plan *plan, int *flags_out) {
    unsigned *h = plan->h_status;
    if (!h || !h[kScalValid]) return BLOCH_OK;
    auto as_float = [](unsigned u) { float f; std::memcpy(&f, &u, sizeof f); return f; };
    int flags = (int)h[kScalFlags];
    const double R = std::sqrt((double)as_float(h[kScalX2Max])), F = (double)as_float(h[kScalDwMax]) / (2.0 * M_PI),
                 V = std::sqrt((double)as_float(h[kScalV2Max]));
    // phase range: only when the phantom exceeds what the plan was told to assume; then the separable bound
    // |k'|max R + F tau_max + |mu'|max V (never below the true worst phase) decides
    double reach = 0.0;
    if (R > plan->ext_m * (1.0 + 1e-6) || F > plan->ext_hz * (1.0 + 1e-6) || V > plan->ext_mps * (1.0 + 1e-6)) {
        reach = plan->k_max * std::max(R, plan->ext_m) + std::max(F, plan->ext_hz) * plan->tau_max +
                plan->m_max * std::max(V, plan->ext_mps);
        const bool fp64 = plan->info.phase_mode == BLOCH_PHASE_FP64;
        if (fp64 ? reach >= kFp64TurnLimit : (plan->phase_requested == BLOCH_PHASE_AUTO && reach > kFp32TurnLimit))
            flags |= BLOCH_STATUS_PHASE_RANGE;
    }
    std::memset(h, 0, kStatusWords * sizeof(unsigned));
    if (flags_out) *flags_out = flags;
    if (flags & (BLOCH_STATUS_BAD_RELAXATION | BLOCH_STATUS_NONFINITE))
        return fail(BLOCH_EINVAL, (flags & BLOCH_STATUS_BAD_RELAXATION)
                                      ? "the phantom holds a T1 or T2 that is <= 0 or not finite"
                                      : "the phantom (or the initial state) holds a non-finite value");
    if (flags & BLOCH_STATUS_PHASE_RANGE) {
        char msg[320];
        std::snprintf(msg, sizeof msg,
                      "phantom outside the plan's phase range: max |x| %.4g m, |dw|/2pi %.4g Hz, |v| %.4g m/s (declared %.4g / "
                      "%.4g / %.4g) give up to %.0f turns per block; create the plan with these extents in bloch_sim_params%s",
                      R, F, V, plan->ext_m, plan->ext_hz, plan->ext_mps, reach,
                      plan->info.phase_mode == BLOCH_PHASE_FP64 ? " and shorter blocks (max_block_points)" : "");
        return fail(BLOCH_ERANGE, msg);
    }
    return BLOCH_OK;
}
}  // namespace bloch

using namespace bloch;

extern "C" {

int bloch_version(void) { return 100; }

const char *bloch_strerror(int code) {
    switch (code) {
        case BLOCH_OK: return "ok";
        case BLOCH_EINVAL: return "invalid argument";
        case BLOCH_ENONMONOTONIC: return "times not ascending or RF samples overlap";
        case BLOCH_EADC_IN_RF: return "ADC sample inside an RF-active run";
        case BLOCH_EWORKSPACE: return "workspace or table buffer too small or misaligned";
        case BLOCH_ECUDA: return "CUDA runtime error";
        case BLOCH_EARCH: return "device is not sm_100";
        case BLOCH_ENOTUPLOADED: return "tables not uploaded";
        case BLOCH_ENOMEM: return "host allocation failed";
        case BLOCH_EHWLIMIT: return "gradient waveform exceeds the scanner's G_max or S_max";
        case BLOCH_ERANGE: return "phantom outside the phase range the plan resolves";
        default: return "unknown error";
    }
}

const char *bloch_last_error(void) { return bloch::last_error_cstr(); }

int bloch_plan_create(const bloch_scanner *scanner, const bloch_sequence *seq, const bloch_sim_params *params,
                      bloch_plan **out) {
    if (!out) return fail(BLOCH_EINVAL, "out is NULL");
    *out = nullptr;
    bloch_plan *p = new (std::nothrow) bloch_plan();
    if (!p) return fail(BLOCH_ENOMEM, "plan allocation failed");
    int rc;
    try {
        rc = build_plan(scanner, seq, params, p);
    } catch (const std::bad_alloc &) {
        rc = fail(BLOCH_ENOMEM, "host allocation failed while planning");
    } catch (...) {
        rc = fail(BLOCH_EINVAL, "unexpected exception while planning");
    }
    if (rc != BLOCH_OK) {
        delete p;
        return rc;
    }
    *out = p;
    return BLOCH_OK;
}

int bloch_plan_destroy(bloch_plan *plan) {
    if (!plan) return BLOCH_OK;
    for (void *e : plan->events) cudaEventDestroy((cudaEvent_t)e);
    if (plan->h_status) cudaFreeHost(plan->h_status);
    delete plan;
    return BLOCH_OK;
}

int bloch_plan_get_info(const bloch_plan *plan, bloch_plan_info *out) {
    if (!plan || !out) return fail(BLOCH_EINVAL, "NULL argument");
    *out = plan->info;
    out->path = plan->path;
    for (int k = 0; k < 16; ++k) out->options[k] = k < BLOCH_N_OPTIONS ? plan->opt[k] : 0;
    return BLOCH_OK;
}

int bloch_plan_host_tables(const bloch_plan *plan, const void **h_tables, size_t *bytes) {
    if (!plan || !h_tables || !bytes) return fail(BLOCH_EINVAL, "NULL argument");
    *h_tables = plan->tables.data();
    *bytes = plan->tables.size();
    return BLOCH_OK;
}

int bloch_plan_workspace_bytes(const bloch_plan *plan, int64_t n_spins, size_t *out) {
    return bloch_plan_workspace_bytes_coils(plan, n_spins, 0, out);
}

int bloch_plan_workspace_bytes_coils(const bloch_plan *plan, int64_t n_spins, int n_coils, size_t *out) {
    if (!plan || !out || n_spins < 0 || n_coils < 0) return fail(BLOCH_EINVAL, "NULL plan/out or negative size");
    if (n_spins > INT32_MAX) return fail(BLOCH_EINVAL, "n_spins exceeds 2^31-1");
    // the current device's SM count -- the number bloch_simulate carves with -- or 148 without a device
    *out = carve(plan, n_spins, nullptr, sm_count_cached(), n_coils).bytes;
    return BLOCH_OK;
}

int bloch_plan_upload(bloch_plan *plan, void *d_tables, size_t bytes, void *stream) {
    if (!plan || !d_tables) return fail(BLOCH_EINVAL, "NULL argument");
    if (bytes < plan->tables.size() || (reinterpret_cast<uintptr_t>(d_tables) % kAlign) != 0)
        return fail(BLOCH_EWORKSPACE, "table buffer too small or not 256-B aligned");
    if (!plan->h_status) {  // 32 B of pinned host memory for the phantom findings (bloch_plan_status)
        BLOCH_CUDA(cudaHostAlloc((void **)&plan->h_status, kStatusWords * sizeof(unsigned), cudaHostAllocDefault));
        std::memset(plan->h_status, 0, kStatusWords * sizeof(unsigned));
    }
    BLOCH_CUDA(cudaMemcpyAsync(d_tables, plan->tables.data(), plan->tables.size(), cudaMemcpyHostToDevice,
                               (cudaStream_t)stream));
    plan->d_tables = (const unsigned char *)d_tables;
    return BLOCH_OK;
}

int bloch_plan_set_profiling(bloch_plan *plan, int enable) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    plan->profiling = enable != 0;
    return BLOCH_OK;
}

int bloch_plan_last_timing(const bloch_plan *plan, float *ms_by_kind, int64_t *launches_by_kind) {
    if (!plan || !ms_by_kind || !launches_by_kind) return fail(BLOCH_EINVAL, "NULL argument");
    for (int k = 0; k < BLOCH_N_KINDS; ++k) {
        ms_by_kind[k] = 0.f;
        launches_by_kind[k] = 0;
    }
    const size_t n = plan->event_kind.size();
    for (size_t k = 0; k + 1 < n; ++k) {
        float ms = 0.f;
        BLOCH_CUDA(cudaEventElapsedTime(&ms, (cudaEvent_t)plan->events[k], (cudaEvent_t)plan->events[k + 1]));
        const int kind = plan->event_kind[k];
        ms_by_kind[kind] += ms;
        launches_by_kind[kind] += 1;
    }
    return BLOCH_OK;
}

int bloch_plan_set_path(bloch_plan *plan, int path) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    if (path != BLOCH_PATH_AUTO && path != BLOCH_PATH_PER_BLOCK && path != BLOCH_PATH_FUSED)
        return fail(BLOCH_EINVAL, "path is not a BLOCH_PATH_* value");
    plan->path = path;
    return BLOCH_OK;
}

int bloch_plan_set_option(bloch_plan *plan, int key, int value) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    bool ok = false;
    switch (key) {
        case BLOCH_OPT_SIGNAL_LIN: case BLOCH_OPT_SIGNAL_FIXED_CTA: ok = value == 0 || value == 1; break;
        case BLOCH_OPT_SIGNAL_P: ok = value == 0 || value == 1 || value == 2 || value == 4 || value == 8; break;
        case BLOCH_OPT_SIGNAL_CTAS_PER_SM: ok = value >= 1 && value <= 8; break;
        case BLOCH_OPT_RF_THREADS: ok = value == 0 || value == 32 || value == 64 || value == 128; break;
        case BLOCH_OPT_RF_SPINS: ok = value >= 0 && value <= 2; break;
        case BLOCH_OPT_COIL_TC: ok = value >= -1 && value <= 2; break;
        case BLOCH_OPT_SEQ_SIG_EXTRA: ok = value >= -1 && value <= 7; break;
        case BLOCH_OPT_SEQ_SIG_BASE: ok = value >= -1 && value <= 7; break;
        case BLOCH_OPT_SEQ_ITEMS_X4: ok = value >= 0 && value <= 64; break;
        case BLOCH_OPT_RF_CONST: ok = value >= 0 && value <= 2; break;
        default: return fail(BLOCH_EINVAL, "unknown BLOCH_OPT_* key");
    }
    if (!ok) return fail(BLOCH_EINVAL, "option value out of range");
    plan->opt[key] = value;
    return BLOCH_OK;
}

int bloch_plan_get_option(const bloch_plan *plan, int key, int *value) {
    if (!plan || !value || key < 0 || key >= BLOCH_N_OPTIONS) return fail(BLOCH_EINVAL, "NULL argument or unknown key");
    *value = plan->opt[key];
    return BLOCH_OK;
}

int bloch_plan_status(const bloch_plan *plan, void *stream, int *flags) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    if (flags) *flags = 0;
    if (!plan->h_status) return BLOCH_OK;  // nothing simulated yet
    BLOCH_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    return bloch::collect_status(plan, flags);
}

int bloch_plan_uses_fused(const bloch_plan *plan, int64_t n_spins, int *out) {
    if (!plan || !out) return fail(BLOCH_EINVAL, "NULL argument");
    const SeqShape q = seq_shape(plan, n_spins, sm_count_cached());
    *out = (q.ok && q.use) ? 1 : 0;
    return BLOCH_OK;
}

int bloch_plan_last_launches(const bloch_plan *plan, int64_t *out) {
    if (!plan || !out) return fail(BLOCH_EINVAL, "NULL argument");
    *out = plan->last.launches;
    return BLOCH_OK;
}

int bloch_plan_last_kernel(const bloch_plan *plan, int kind, char *name, size_t name_bytes, int64_t *grid_ctas,
                           int *block_threads) {
    if (!plan || kind < 0 || kind >= BLOCH_N_KINDS) return fail(BLOCH_EINVAL, "NULL plan or bad kind");
    const KernelNote &k = plan->last_kernel[kind];
    if (name && name_bytes > 0) {
        std::strncpy(name, k.name, name_bytes - 1);
        name[name_bytes - 1] = 0;
    }
    if (grid_ctas) *grid_ctas = k.grid;
    if (block_threads) *block_threads = k.block;
    return BLOCH_OK;
}

int bloch_simulate(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                   const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                   const float *d_dw, float *d_Mxy, float *d_Mz, int init_equilibrium, float *d_signal,
                   void *d_workspace, size_t workspace_bytes, void *stream_) {
    return bloch_simulate_motion(plan, n_spins, d_x, d_y, d_z, d_M0, d_T1, d_T2, d_dw, nullptr, nullptr, nullptr, d_Mxy,
                                 d_Mz, init_equilibrium, d_signal, d_workspace, workspace_bytes, stream_);
}

namespace bloch {
namespace {
int simulate_impl(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                  const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                  const float *d_dw, const float *d_vx, const float *d_vy, const float *d_vz,
                  int n_coils, const float *d_coil,
                  float *d_Mxy, float *d_Mz, int init_equilibrium, float *d_signal,
                  void *d_workspace, size_t workspace_bytes, void *stream_);
}
}  // namespace bloch

int bloch_simulate_motion(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                          const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                          const float *d_dw, const float *d_vx, const float *d_vy, const float *d_vz,
                          float *d_Mxy, float *d_Mz, int init_equilibrium, float *d_signal,
                          void *d_workspace, size_t workspace_bytes, void *stream_) {
    return bloch::simulate_impl(plan, n_spins, d_x, d_y, d_z, d_M0, d_T1, d_T2, d_dw, d_vx, d_vy, d_vz, 0, nullptr,
                                d_Mxy, d_Mz, init_equilibrium, d_signal, d_workspace, workspace_bytes, stream_);
}

int bloch_simulate_coils(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                         const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                         const float *d_dw, int n_coils, const float *d_coil, float *d_Mxy, float *d_Mz,
                         int init_equilibrium, float *d_signal, void *d_workspace, size_t workspace_bytes,
                         void *stream_) {
    return bloch_simulate_coils_motion(plan, n_spins, d_x, d_y, d_z, d_M0, d_T1, d_T2, d_dw, nullptr, nullptr, nullptr,
                                       n_coils, d_coil, d_Mxy, d_Mz, init_equilibrium, d_signal, d_workspace,
                                       workspace_bytes, stream_);
}

int bloch_simulate_coils_motion(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                                const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                                const float *d_dw, const float *d_vx, const float *d_vy, const float *d_vz, int n_coils,
                                const float *d_coil, float *d_Mxy, float *d_Mz, int init_equilibrium, float *d_signal,
                                void *d_workspace, size_t workspace_bytes, void *stream_) {
    if (!plan) return bloch::fail(BLOCH_EINVAL, "NULL plan");
    if (n_coils < 1 || n_coils > 4096) return bloch::fail(BLOCH_EINVAL, "n_coils must be in [1, 4096]");
    if (n_spins > 0 && !d_coil) return bloch::fail(BLOCH_EINVAL, "d_coil is NULL");
    if (plan->info.output_mode != BLOCH_OUT_SUM_ALL)
        return bloch::fail(BLOCH_EINVAL, "multi-coil receive needs a BLOCH_OUT_SUM_ALL plan");
    return bloch::simulate_impl(plan, n_spins, d_x, d_y, d_z, d_M0, d_T1, d_T2, d_dw, d_vx, d_vy, d_vz, n_coils,
                                d_coil, d_Mxy, d_Mz, init_equilibrium, d_signal, d_workspace, workspace_bytes, stream_);
}

namespace bloch {
namespace {
int simulate_impl(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                  const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                  const float *d_dw, const float *d_vx, const float *d_vy, const float *d_vz,
                  int n_coils, const float *d_coil,
                  float *d_Mxy, float *d_Mz, int init_equilibrium, float *d_signal,
                  void *d_workspace, size_t workspace_bytes, void *stream_) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    const bool has_v = d_vx || d_vy || d_vz;
    if (has_v && !(d_vx && d_vy && d_vz)) return fail(BLOCH_EINVAL, "give all of d_vx, d_vy, d_vz or none");
    if (has_v && plan->info.motion_mode == BLOCH_MOTION_NONE)
        return fail(BLOCH_EINVAL, "velocities given but the plan was created without motion (BLOCH_MOTION_LINEAR / _WAVEFORM)");
    const bool mo = plan->info.motion_mode != BLOCH_MOTION_NONE;
    if (n_spins < 0 || n_spins > INT32_MAX) return fail(BLOCH_EINVAL, "n_spins out of range");
    if (!plan->d_tables) return fail(BLOCH_ENOTUPLOADED, "call bloch_plan_upload first");
    if (n_spins > 0 && (!d_x || !d_y || !d_z || !d_M0 || !d_T1 || !d_T2 || !d_dw))
        return fail(BLOCH_EINVAL, "NULL phantom array");
    if (!init_equilibrium && (!d_Mxy || !d_Mz)) return fail(BLOCH_EINVAL, "initial state requested but d_Mxy/d_Mz NULL");
    if ((d_Mxy == nullptr) != (d_Mz == nullptr)) return fail(BLOCH_EINVAL, "d_Mxy and d_Mz must both be given or both NULL");
    if (plan->info.n_adc > 0 && !d_signal) return fail(BLOCH_EINVAL, "d_signal is NULL");
    int rc = check_arch();
    if (rc != BLOCH_OK) return rc;
    // findings of an earlier simulation on this plan that nobody collected (bloch_plan_status): fail now, once
    if (plan->h_status && plan->h_status[kScalValid] && (rc = collect_status(plan, nullptr)) != BLOCH_OK) return rc;
    const int sms = sm_count_cached();
    cudaStream_t stream = (cudaStream_t)stream_;
    const bool grouped = plan->info.output_mode == BLOCH_OUT_GROUPED;
    const bool per_spin = plan->info.output_mode == BLOCH_OUT_PER_SPIN || grouped;  // no cross-CTA reduction
    if (grouped && n_spins % plan->info.group_size != 0)
        return fail(BLOCH_EINVAL, "n_spins is not a multiple of the plan's group_size");
    const bool ph64 = plan->info.phase_mode == BLOCH_PHASE_FP64;

    if (n_spins == 0) {  // degenerate: the sum over no spins is zero
        if (!per_spin && plan->info.n_adc > 0)
            BLOCH_CUDA(cudaMemsetAsync(d_signal, 0, size_t(std::max(n_coils, 1)) * size_t(plan->info.n_adc) * sizeof(float2),
                                       stream));
        return BLOCH_OK;
    }
    if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) % kAlign) != 0)
        return fail(BLOCH_EWORKSPACE, "workspace NULL or not 256-B aligned");
    const Workspace w = carve(plan, n_spins, d_workspace, sms, n_coils);
    if (workspace_bytes < w.bytes) return fail(BLOCH_EWORKSPACE, "workspace too small; see bloch_plan_workspace_bytes[_coils]");

    const int n = (int)n_spins;
    for (KernelNote &k : plan->last_kernel) k = KernelNote{};
    Taps taps{plan, stream};
    int64_t launches = 0;
    if ((rc = taps.mark(BLOCH_KIND_OTHER))) return rc;
    BLOCH_CUDA(cudaMemsetAsync(w.scal, 0, kAlign, stream));
    pack_kernel<<<(n + 255) / 256, 256, 0, stream>>>(n, d_x, d_y, d_z, d_M0, d_T1, d_T2, d_dw,
                                                     (const float2 *)d_Mxy, d_Mz, init_equilibrium ? 1 : 0,
                                                     w.A, w.C, w.S, w.Ad, w.scal, d_vx, d_vy, d_vz, w.V, w.Vd);
    ++launches;
    const bool coil_fused = coil_use_fused(plan, n_spins, sms, n_coils);
    const bool tc = n_coils > 0 && !coil_fused && coil_use_tc(plan, n_spins, n_coils);
    const int ncp = tc ? tc_coils_per_pass(n_coils) : coils_per_pass(n_coils);
    const int n_pass = (n_coils + ncp - 1) / ncp;
    const int n_pad = (n + kTcStageSpins - 1) / kTcStageSpins * kTcStageSpins;
    DeviceInfo *devinfo = current_device();  // non-NULL: check_arch passed
    const bool tc_h = tc && coil_tc_fp16(plan);
    if (tc_h) {
        if (!devinfo->h_attr.load(std::memory_order_acquire)) {  // once per DEVICE (the attribute is per device)
            BLOCH_CUDA(cudaFuncSetAttribute(signal_coils_h_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h_smem(8)));
            BLOCH_CUDA(cudaFuncSetAttribute(signal_coils_h_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h_smem(16)));
            BLOCH_CUDA(cudaFuncSetAttribute(signal_coils_h_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h_smem(32)));
            devinfo->h_attr.store(true, std::memory_order_release);
        }
        // operand scales from measured maxima (scal[6], scal[7]; cleared with the findings word above), then the B tiles
        coil_scales_kernel<<<std::min(4 * sms, (n + 255) / 256 * std::max(n_coils, 1)), 256, 0, stream>>>(
            n, w.C, w.S, (const float2 *)d_coil, (long long)n_coils * n, w.scal);
        const dim3 pg((n_pad + 255) / 256, n_pass);
        if (ncp == 32) pack_coils_h_kernel<32><<<pg, 256, 0, stream>>>(n, n_pad, n_coils, (const float2 *)d_coil, w.scal, (unsigned char *)w.W);
        else if (ncp == 16) pack_coils_h_kernel<16><<<pg, 256, 0, stream>>>(n, n_pad, n_coils, (const float2 *)d_coil, w.scal, (unsigned char *)w.W);
        else pack_coils_h_kernel<8><<<pg, 256, 0, stream>>>(n, n_pad, n_coils, (const float2 *)d_coil, w.scal, (unsigned char *)w.W);
        launches += 2;
    } else if (tc) {
        if (!devinfo->tc_attr.load(std::memory_order_acquire)) {  // once per DEVICE (the attribute is per device)
            BLOCH_CUDA(cudaFuncSetAttribute(signal_coils_tc_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_smem(8)));
            BLOCH_CUDA(cudaFuncSetAttribute(signal_coils_tc_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_smem(16)));
            BLOCH_CUDA(cudaFuncSetAttribute(signal_coils_tc_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_smem(32)));
            devinfo->tc_attr.store(true, std::memory_order_release);
        }
        const dim3 pg((n_pad + 255) / 256, n_pass);
        if (ncp == 32) pack_coils_tc_kernel<32><<<pg, 256, 0, stream>>>(n, n_pad, n_coils, (const float2 *)d_coil, (unsigned char *)w.W);
        else if (ncp == 16) pack_coils_tc_kernel<16><<<pg, 256, 0, stream>>>(n, n_pad, n_coils, (const float2 *)d_coil, (unsigned char *)w.W);
        else pack_coils_tc_kernel<8><<<pg, 256, 0, stream>>>(n, n_pad, n_coils, (const float2 *)d_coil, (unsigned char *)w.W);
        ++launches;
    } else if (n_coils > 0) {
        pack_coils_kernel<<<dim3((n + 255) / 256, n_pass), 256, 0, stream>>>(n, n_coils, ncp, (const float2 *)d_coil, w.W);
        ++launches;
    }

    const SeqShape sq = seq_shape(plan, n_spins, sms, n_coils);  // coils: up to 8 inside the launch, else per-block
    if (plan->path == BLOCH_PATH_FUSED && !sq.ok)
        return fail(BLOCH_EINVAL, "BLOCH_PATH_FUSED needs SUM_ALL output (or PER_SPIN with <= 16 samples per block), fp32 phase, no motion, <= 29 x 32 spins per SM and <= 8 receive coils");
    if (sq.ok && sq.use) {
        // ONE persistent launch for the whole sequence + the second pass over all ADC samples
        if (!devinfo->seq_attr.load(std::memory_order_acquire)) {  // once per DEVICE; sticky for the function there
            BLOCH_CUDA(cudaFuncSetAttribute(seq_kernel<false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)seq_smem_bytes(kSeqMaxThreads)));
            BLOCH_CUDA(cudaFuncSetAttribute(seq_kernel<true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)seq_smem_bytes(kSeqMaxThreads)));
            BLOCH_CUDA(cudaFuncSetAttribute(seq_kernel<false, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)seq_smem_bytes(kSeqMaxThreads, 4)));
            BLOCH_CUDA(cudaFuncSetAttribute(seq_kernel<false, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)seq_smem_bytes(kSeqMaxThreads, 8)));
            devinfo->seq_attr.store(true, std::memory_order_release);
        }
        if ((rc = taps.mark(BLOCH_KIND_FUSED))) return rc;
        const SeqOp *prog = reinterpret_cast<const SeqOp *>(plan->d_tables + plan->prog_off);
        note_kernel(plan, BLOCH_KIND_FUSED, sq.n_ctas, sq.threads, "seq_kernel<%d, %d>", per_spin ? 1 : 0, sq.nc);
        // kernel arguments by address (cudaLaunchCooperativeKernel)
        const unsigned char *a_tables = plan->d_tables;
        int a_nops = (int)plan->blocks.size(), a_n = n, a_chunk = sq.chunk, a_rfw = sq.rf_warps, a_min = sq.min_items;
        const float4 *a_A = w.A, *a_C = w.C;
        float4 *a_S = w.S;
        SeqRoles a_roles = sq.roles;
        const float *a_scal = (const float *)w.scal;
        float2 *a_ring = w.partial;
        int a_slots = sq.ring_slots, a_stride = sq.slot_stride, a_nblk = (int)plan->n_adc_blocks;
        int *a_tickets = reinterpret_cast<int *>(w.partial + sq.ticket_off);
        const SeqAdcBlock *a_blk = reinterpret_cast<const SeqAdcBlock *>(plan->d_tables + plan->adcblk_off);
        float2 *a_sig = per_spin ? nullptr : (float2 *)d_signal, *a_ps = per_spin ? (float2 *)d_signal : nullptr;
        long long a_nadc = (long long)plan->info.n_adc;
        int a_final = d_Mxy ? 1 : 0;
        const float4 *a_W = reinterpret_cast<const float4 *>(w.W);  // coils: nc float2 per spin (pack_coils_kernel, one pass)
        int a_ncoils = n_coils;
        void *args[] = {&a_tables, &prog, &a_nops, &a_A, &a_C, &a_S, &a_n, &a_chunk, &a_rfw, &a_roles, &a_min, &a_scal,
                        &a_ring, &a_slots, &a_stride, &a_tickets, &a_nblk, &a_blk, &a_sig, &a_nadc, &a_final, &a_ps,
                        &a_W, &a_ncoils};
        if (per_spin) {
            BLOCH_CUDA(cudaLaunchKernel((const void *)seq_kernel<true, 0>, dim3(sq.n_ctas), dim3(sq.threads), args, sq.smem, stream));
        } else {
            // the CTAs wait for one another's tickets (integer counters) when they sum the partial rows, so all of them
            // must be resident: a cooperative launch guarantees it (n_ctas <= SMs, one CTA per SM)
            BLOCH_CUDA(cudaMemsetAsync(a_tickets, 0, size_t(2) * size_t(std::max(a_nblk, 1)) * sizeof(int), stream));
            const void *fn = sq.nc == 8 ? (const void *)seq_kernel<false, 8>
                                        : (sq.nc == 4 ? (const void *)seq_kernel<false, 4> : (const void *)seq_kernel<false, 0>);
            BLOCH_CUDA(cudaLaunchCooperativeKernel(fn, dim3(sq.n_ctas), dim3(sq.threads), args, sq.smem, stream));
        }
        ++launches;
        if (d_Mxy) {
            if ((rc = taps.mark(BLOCH_KIND_OTHER))) return rc;
            unpack_kernel<<<(n + 255) / 256, 256, 0, stream>>>(n, w.S, (float2 *)d_Mxy, d_Mz);
            ++launches;
        }
        if ((rc = taps.mark(BLOCH_KIND_OTHER))) return rc;  // closing event
        if (plan->profiling) plan->event_kind.resize(taps.used);
        plan->last.launches = launches;
        BLOCH_CUDA(cudaGetLastError());
        // what pack_kernel found out about the phantom follows the simulation to the host (bloch_plan_status)
        BLOCH_CUDA(cudaMemcpyAsync(plan->h_status, w.scal, kStatusWords * sizeof(unsigned), cudaMemcpyDeviceToHost, stream));
        return BLOCH_OK;
    }

    bool pending = false;
    PropRec prop{0, 0, 0, 0, 0, 0, 0};
    // RF launch shape: one spin per thread; small CTAs when spins are few so the warps spread over all
    // 592 sub-partitions, 128-thread CTAs once there are >= 32 warps per SM
    // two spins per thread (rf_pair_kernel; static plans) on request: measured in DESIGN.md section 12
    const bool rf_pair = !mo && plan->opt[BLOCH_OPT_RF_SPINS] == 2;
    const int rf_items = rf_pair ? (n + 1) / 2 : n;
    const int rf_threads = plan->opt[BLOCH_OPT_RF_THREADS] ? plan->opt[BLOCH_OPT_RF_THREADS]
                                                           : ((rf_items + 31) / 32 >= sms * 32 ? 128 : 32);
    const int rf_grid = (rf_items + rf_threads - 1) / rf_threads;
    auto launch_rf = [&](const unsigned char *tbl, int n_tiles, int has_prop) -> int {
        if (tbl) note_kernel(plan, BLOCH_KIND_RF, rf_grid, rf_threads, rf_pair ? "rf_pair_kernel" : "rf_kernel<%d>", mo ? 1 : 0);
        if (rf_pair) rf_pair_kernel<<<rf_grid, rf_threads, 0, stream>>>(tbl, n_tiles, prop, has_prop, w.A, w.C, w.S, n);
        else if (mo) rf_kernel<true><<<rf_grid, rf_threads, 0, stream>>>(tbl, n_tiles, prop, has_prop, w.A, w.C, w.S, w.V, n);
        else rf_kernel<false><<<rf_grid, rf_threads, 0, stream>>>(tbl, n_tiles, prop, has_prop, w.A, w.C, w.S, nullptr, n);
        return BLOCH_OK;
    };
    bool batch_open = false;
    SigShape batch_shape{};
    int64_t batch_adc_first = 0, batch_pts = 0, batch_done = 0;
    for (size_t bi = 0; bi < plan->blocks.size(); ++bi) {
        const Block &b = plan->blocks[bi];
        if (b.type == kBlockRF) {
            if ((rc = taps.mark(BLOCH_KIND_RF))) return rc;
            // (from 16,384 spins on: below that the launch is latency-bound and the 25 KB of parameters cost 2-3 us)
            if (b.rf_const_count > 0 && !mo && !rf_pair &&
                (plan->opt[BLOCH_OPT_RF_CONST] == 2 || (plan->opt[BLOCH_OPT_RF_CONST] == 1 && n >= 16384))) {
                // the block's step records by value, as kernel parameters (plan.cpp): rf_const_kernel, bitwise rf_kernel
                for (int64_t c = 0; c < b.rf_const_count; ++c) {
                    if (c > 0 && (rc = taps.mark(BLOCH_KIND_RF))) return rc;
                    rf_const_kernel<<<rf_grid, rf_threads, 0, stream>>>(plan->rf_const[size_t(b.rf_const_first + c)], prop,
                                                                        (c == 0 && pending) ? 1 : 0, w.A, w.C, w.S, n);
                    ++launches;
                }
                note_kernel(plan, BLOCH_KIND_RF, rf_grid, rf_threads, "rf_const_kernel");
                pending = false;
                continue;
            }
            if ((rc = launch_rf(plan->d_tables + b.table_off, (int)b.n_tiles, pending ? 1 : 0))) return rc;
            ++launches;
            pending = false;
            continue;
        }
        if (pending) {  // two precession blocks in a row: apply the first one's end transform now
            if ((rc = taps.mark(BLOCH_KIND_OTHER))) return rc;
            if ((rc = launch_rf(nullptr, 0, 1))) return rc;
            ++launches;
            pending = false;
        }
        if (b.adc_count > 0) {
            if ((rc = taps.mark(BLOCH_KIND_SIGNAL))) return rc;
            const void *recs = plan->d_tables + b.table_off;
            const int n_pts = (int)b.adc_count;
            if (grouped) {
                const int gs = plan->info.group_size, n_groups = n / gs;
                const unsigned grid = (unsigned)(((long long)n_groups * 32 + 255) / 256);
                if (ph64)
                    grouped_kernel<true><<<grid, 256, 0, stream>>>(recs, n_pts, w.A, w.C, w.S, w.V, n_groups, gs,
                                                                   (long long)plan->info.n_adc, (long long)b.adc_first,
                                                                   (float2 *)d_signal);
                else
                    grouped_kernel<false><<<grid, 256, 0, stream>>>(recs, n_pts, w.A, w.C, w.S, w.V, n_groups, gs,
                                                                    (long long)plan->info.n_adc, (long long)b.adc_first,
                                                                    (float2 *)d_signal);
                note_kernel(plan, BLOCH_KIND_SIGNAL, grid, 256, "grouped_kernel<%d>", ph64 ? 1 : 0);
                ++launches;
            } else if (per_spin) {
                const long long total = (long long)n * n_pts;
                const unsigned grid = (unsigned)((total + 255) / 256);
                if (ph64)
                    perspin_kernel<true><<<grid, 256, 0, stream>>>(recs, n_pts, w.A, w.C, w.S, w.V, n,
                                                                   (long long)plan->info.n_adc, (long long)b.adc_first,
                                                                   (float2 *)d_signal);
                else
                    perspin_kernel<false><<<grid, 256, 0, stream>>>(recs, n_pts, w.A, w.C, w.S, w.V, n,
                                                                    (long long)plan->info.n_adc, (long long)b.adc_first,
                                                                    (float2 *)d_signal);
                note_kernel(plan, BLOCH_KIND_SIGNAL, grid, 256, "perspin_kernel<%d>", ph64 ? 1 : 0);
                ++launches;
            } else if (n_coils > 0) {
                const SigShape s = coil_shape(n_pts, n, sms, ncp, tc);
                const dim3 grid(s.ptiles, s.chunks);
                for (int pass = 0; pass < n_pass; ++pass) {
                    const float4 *Wp = reinterpret_cast<const float4 *>(w.W + (size_t)pass * n * ncp);
                    const int in_pass = std::min(ncp, n_coils - pass * ncp);
                    if (pass > 0 && (rc = taps.mark(BLOCH_KIND_SIGNAL))) return rc;
#define BLOCH_LAUNCH_COIL(PP, NCC, H, M, AP, VP)                                                                       \
    signal_coils_kernel<PP, NCC, H, M><<<grid, s.threads, 0, stream>>>(recs, n_pts, AP, VP, w.S, Wp, n, s.spins_per_chunk, \
                                                                         (const float *)w.scal, w.partial)
#define BLOCH_LAUNCH_COIL2(PP, NCC)                                        \
    do {                                                                   \
        if (ph64 && mo) BLOCH_LAUNCH_COIL(PP, NCC, true, true, w.Ad, w.Vd);    \
        else if (ph64) BLOCH_LAUNCH_COIL(PP, NCC, true, false, w.Ad, nullptr); \
        else if (mo) BLOCH_LAUNCH_COIL(PP, NCC, false, true, w.A, w.V);        \
        else BLOCH_LAUNCH_COIL(PP, NCC, false, false, w.A, nullptr);           \
    } while (0)
                    if (tc) note_kernel(plan, BLOCH_KIND_SIGNAL, (int64_t)grid.x * grid.y, kTcThreads,
                                        tc_h ? "signal_coils_h_kernel<%d>" : "signal_coils_tc_kernel<%d>", ncp);
                    else note_kernel(plan, BLOCH_KIND_SIGNAL, (int64_t)grid.x * grid.y, s.threads, "signal_coils_kernel<%d, %d, %d, %d>",
                                     s.P == 2 ? 2 : 1, ncp == 8 ? 8 : 4, ph64 ? 1 : 0, mo ? 1 : 0);
                    if (tc_h) {
                        if (pass == 0) {  // this block's start states in polar form, once for all passes
                            coil_polar_kernel<<<(n + 255) / 256, 256, 0, stream>>>(n, w.S, w.Sp);
                            ++launches;
                        }
                        const unsigned char *Bp = (const unsigned char *)w.W + (size_t)pass * (n_pad / 8) * h_btile(ncp);
                        if (ncp == 32)
                            signal_coils_h_kernel<32><<<grid, kTcThreads, h_smem(32), stream>>>(
                                (const float4 *)recs, n_pts, w.A, w.Sp, Bp, n, s.spins_per_chunk, w.scal, w.partial);
                        else if (ncp == 16)
                            signal_coils_h_kernel<16><<<grid, kTcThreads, h_smem(16), stream>>>(
                                (const float4 *)recs, n_pts, w.A, w.Sp, Bp, n, s.spins_per_chunk, w.scal, w.partial);
                        else
                            signal_coils_h_kernel<8><<<grid, kTcThreads, h_smem(8), stream>>>(
                                (const float4 *)recs, n_pts, w.A, w.Sp, Bp, n, s.spins_per_chunk, w.scal, w.partial);
                    } else if (tc) {
                        const unsigned char *Bp = (const unsigned char *)w.W + (size_t)pass * (n_pad / 8) * tc_bgroup(ncp);
                        if (ncp == 32)
                            signal_coils_tc_kernel<32><<<grid, kTcThreads, tc_smem(32), stream>>>(
                                (const float4 *)recs, n_pts, w.A, w.S, Bp, n, s.spins_per_chunk, (const float *)w.scal, w.partial);
                        else if (ncp == 16)
                            signal_coils_tc_kernel<16><<<grid, kTcThreads, tc_smem(16), stream>>>(
                                (const float4 *)recs, n_pts, w.A, w.S, Bp, n, s.spins_per_chunk, (const float *)w.scal, w.partial);
                        else
                            signal_coils_tc_kernel<8><<<grid, kTcThreads, tc_smem(8), stream>>>(
                                (const float4 *)recs, n_pts, w.A, w.S, Bp, n, s.spins_per_chunk, (const float *)w.scal, w.partial);
                    }
                    else if (ncp == 8) { if (s.P == 2) BLOCH_LAUNCH_COIL2(2, 8); else BLOCH_LAUNCH_COIL2(1, 8); }
                    else { if (s.P == 2) BLOCH_LAUNCH_COIL2(2, 4); else BLOCH_LAUNCH_COIL2(1, 4); }
#undef BLOCH_LAUNCH_COIL2
#undef BLOCH_LAUNCH_COIL
                    if ((rc = taps.mark(BLOCH_KIND_REDUCE))) return rc;
                    reduce_coils_kernel<<<dim3((unsigned)((n_pts + 31) / 32), in_pass), dim3(32, 8), 0, stream>>>(
                        w.partial, s.chunks, n_pts,
                        (float2 *)d_signal + (size_t)pass * ncp * (size_t)plan->info.n_adc + b.adc_first,
                        (long long)plan->info.n_adc);
                    launches += 2;
                }
            } else {
                const SigShape s = block_shape(plan, b, n, sms);
                if (!batch_open) {  // look ahead: how many of the following blocks share this batch
                    batch_shape = s;
                    batch_adc_first = b.adc_first;
                    batch_pts = 0;
                    batch_done = 0;
                    const int64_t cap_pts = std::max<int64_t>(n_pts, (int64_t)(w.partial_elems / (size_t)s.chunks));
                    for (size_t bj = bi; bj < plan->blocks.size(); ++bj) {
                        const Block &c = plan->blocks[bj];
                        if (c.type != kBlockPrecession || c.adc_count == 0) continue;
                        const SigShape sc = block_shape(plan, c, n, sms);
                        if (sc.P != s.P || sc.chunks != s.chunks || sc.spins_per_chunk != s.spins_per_chunk ||
                            sc.threads != s.threads) break;
                        if (batch_pts + c.adc_count > cap_pts || batch_pts + c.adc_count > INT32_MAX) break;
                        batch_pts += c.adc_count;
                    }
                    batch_open = true;
                }
                const dim3 grid(s.ptiles, s.chunks);
                const int row = (int)batch_pts, poff = (int)batch_done;
                const int allow_lin = plan->opt[BLOCH_OPT_SIGNAL_LIN];
#define BLOCH_LAUNCH_SIG3(PP, H, M, AP, VP)                                                                    \
    signal_kernel<PP, H, M><<<grid, s.threads, 0, stream>>>(recs, n_pts, AP, VP, w.S, n, s.spins_per_chunk,    \
                                                              (const float *)w.scal, w.partial, row, poff, allow_lin)
#define BLOCH_LAUNCH_SIG(PP)                                                                                   \
    do {                                                                                                       \
        if (ph64 && mo) BLOCH_LAUNCH_SIG3(PP, true, true, w.Ad, w.Vd);                                         \
        else if (ph64) BLOCH_LAUNCH_SIG3(PP, true, false, w.Ad, nullptr);                                      \
        else if (mo) BLOCH_LAUNCH_SIG3(PP, false, true, w.A, w.V);                                             \
        else BLOCH_LAUNCH_SIG3(PP, false, false, w.A, nullptr);                                                \
    } while (0)
                if (b.lin_pts > 0 && allow_lin)
                    note_kernel(plan, BLOCH_KIND_SIGNAL, (int64_t)grid.x * grid.y, s.threads, "signal_lin_kernel<%d, %d>", ph64 ? 1 : 0, mo ? 1 : 0);
                else
                    note_kernel(plan, BLOCH_KIND_SIGNAL, (int64_t)grid.x * grid.y, s.threads, "signal_kernel<%d, %d, %d>", s.P, ph64 ? 1 : 0, mo ? 1 : 0);
                if (b.lin_pts > 0 && allow_lin) {
                    // Cartesian readout (planner: constant k' step, quadratic mu', inside every aligned group of kLinP
                    // samples): the recurrence kernel on the first lin_pts samples, the n % kLinP tail through
                    // signal_kernel<1>; both with this block's chunking, so the partial rows and the second pass are unchanged
                    const int n_groups = (int)(b.lin_pts / kLinP);
                    const dim3 lgrid(s.ptiles, s.chunks);
                    const int n_tail = n_pts - (int)b.lin_pts;
                    const void *trecs = (const unsigned char *)recs + (size_t)b.lin_pts * (ph64 ? 32 : 16) * (mo ? 2 : 1);
                    const dim3 tgrid(1, s.chunks);
                    const int toff = poff + (int)b.lin_pts;
#define BLOCH_LAUNCH_LIN(H, M, AP, VP)                                                                              \
    do {                                                                                                            \
        signal_lin_kernel<H, M><<<lgrid, s.threads, 0, stream>>>(recs, n_groups, AP, VP, w.S, n, s.spins_per_chunk, \
                                                                   (const float *)w.scal, w.partial, row, poff);    \
        if (n_tail > 0)                                                                                             \
            signal_kernel<1, H, M><<<tgrid, 32, 0, stream>>>(trecs, n_tail, AP, VP, w.S, n, s.spins_per_chunk,      \
                                                             (const float *)w.scal, w.partial, row, toff, 0);       \
    } while (0)
                    if (ph64 && mo) BLOCH_LAUNCH_LIN(true, true, w.Ad, w.Vd);
                    else if (ph64) BLOCH_LAUNCH_LIN(true, false, w.Ad, nullptr);
                    else if (mo) BLOCH_LAUNCH_LIN(false, true, w.A, w.V);
                    else BLOCH_LAUNCH_LIN(false, false, w.A, nullptr);
#undef BLOCH_LAUNCH_LIN
                    if (n_tail > 0) ++launches;
                }
                else if (s.P == 8) BLOCH_LAUNCH_SIG(8);
                else if (s.P == 4) BLOCH_LAUNCH_SIG(4);
                else if (s.P == 2) BLOCH_LAUNCH_SIG(2);
                else BLOCH_LAUNCH_SIG(1);
#undef BLOCH_LAUNCH_SIG
#undef BLOCH_LAUNCH_SIG3
                ++launches;
                batch_done += n_pts;
                if (batch_done == batch_pts) {  // batch complete: second pass over all its points
                    if ((rc = taps.mark(BLOCH_KIND_REDUCE))) return rc;
                    reduce_kernel<<<(unsigned)((batch_pts + 31) / 32), dim3(32, 8), 0, stream>>>(
                        w.partial, batch_shape.chunks, (int)batch_pts, (float2 *)d_signal + batch_adc_first);
                    ++launches;
                    batch_open = false;
                }
            }
        }
        prop.kx = b.kend[0];
        prop.ky = b.kend[1];
        prop.kz = b.kend[2];
        prop.tau = b.tau_end;
        prop.mx = b.mend[0];
        prop.my = b.mend[1];
        prop.mz = b.mend[2];
        pending = b.count > 0;  // an empty block (an ADC sample inside an RF run) has nothing to propagate
    }
    if (d_Mxy) {
        if (pending) {
            if ((rc = taps.mark(BLOCH_KIND_OTHER))) return rc;
            if ((rc = launch_rf(nullptr, 0, 1))) return rc;
            ++launches;
        }
        if ((rc = taps.mark(BLOCH_KIND_OTHER))) return rc;
        unpack_kernel<<<(n + 255) / 256, 256, 0, stream>>>(n, w.S, (float2 *)d_Mxy, d_Mz);
        ++launches;
    }
    if ((rc = taps.mark(BLOCH_KIND_OTHER))) return rc;  // closing event
    if (plan->profiling) plan->event_kind.resize(taps.used);
    plan->last.launches = launches;
    BLOCH_CUDA(cudaGetLastError());
    BLOCH_CUDA(cudaMemcpyAsync(plan->h_status, w.scal, kStatusWords * sizeof(unsigned), cudaMemcpyDeviceToHost, stream));
    return BLOCH_OK;
}
}  // namespace
}  // namespace bloch

int bloch_simulate_host_scratch_bytes(const bloch_plan *plan, int64_t n_spins, size_t *out) {
    if (!plan || !out || n_spins < 0) return fail(BLOCH_EINVAL, "NULL plan/out or negative n_spins");
    size_t ws = 0;
    int rc = bloch_plan_workspace_bytes(plan, n_spins, &ws);
    if (rc) return rc;
    const size_t arr = align_up(size_t(n_spins) * sizeof(float), kAlign);
    const size_t sig = signal_rows(plan, n_spins) * size_t(plan->info.n_adc) * sizeof(float2);
    *out = 13 * arr + align_up(sig, kAlign) + ws + kAlign;
    return BLOCH_OK;
}

int bloch_simulate_host(const bloch_plan *plan, int64_t n_spins, const float *h_x, const float *h_y,
                        const float *h_z, const float *h_M0, const float *h_T1, const float *h_T2,
                        const float *h_dw, float *h_Mxy, float *h_Mz, int init_equilibrium, float *h_signal,
                        void *d_scratch, size_t scratch_bytes, void *stream_) {
    return bloch_simulate_host_motion(plan, n_spins, h_x, h_y, h_z, h_M0, h_T1, h_T2, h_dw, nullptr, nullptr, nullptr,
                                      h_Mxy, h_Mz, init_equilibrium, h_signal, d_scratch, scratch_bytes, stream_);
}

int bloch_simulate_host_motion(const bloch_plan *plan, int64_t n_spins, const float *h_x, const float *h_y,
                               const float *h_z, const float *h_M0, const float *h_T1, const float *h_T2,
                               const float *h_dw, const float *h_vx, const float *h_vy, const float *h_vz,
                               float *h_Mxy, float *h_Mz, int init_equilibrium, float *h_signal,
                               void *d_scratch, size_t scratch_bytes, void *stream_) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    const bool has_v = h_vx || h_vy || h_vz;
    if (has_v && !(h_vx && h_vy && h_vz)) return fail(BLOCH_EINVAL, "give all of h_vx, h_vy, h_vz or none");
    size_t need = 0;
    int rc = bloch_simulate_host_scratch_bytes(plan, n_spins, &need);
    if (rc) return rc;
    if (!d_scratch || scratch_bytes < need || (reinterpret_cast<uintptr_t>(d_scratch) % kAlign) != 0)
        return fail(BLOCH_EWORKSPACE, "scratch NULL, too small or not 256-B aligned");
    if (n_spins > 0 && (!h_x || !h_y || !h_z || !h_M0 || !h_T1 || !h_T2 || !h_dw))
        return fail(BLOCH_EINVAL, "NULL phantom array");
    if (!init_equilibrium && (!h_Mxy || !h_Mz)) return fail(BLOCH_EINVAL, "initial state requested but h_Mxy/h_Mz NULL");
    if ((h_Mxy == nullptr) != (h_Mz == nullptr)) return fail(BLOCH_EINVAL, "h_Mxy and h_Mz must both be given or both NULL");
    if (plan->info.n_adc > 0 && !h_signal) return fail(BLOCH_EINVAL, "h_signal is NULL");
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t arr = align_up(size_t(n_spins) * sizeof(float), kAlign);
    unsigned char *base = (unsigned char *)d_scratch;
    float *d[7];
    const float *h[7] = {h_x, h_y, h_z, h_M0, h_T1, h_T2, h_dw};
    for (int k = 0; k < 7; ++k) {
        d[k] = (float *)(base + k * arr);
        if (n_spins > 0)
            BLOCH_CUDA(cudaMemcpyAsync(d[k], h[k], size_t(n_spins) * sizeof(float), cudaMemcpyHostToDevice, stream));
    }
    float *d_Mxy = h_Mxy ? (float *)(base + 7 * arr) : nullptr;
    float *d_Mz = h_Mz ? (float *)(base + 9 * arr) : nullptr;
    if (!init_equilibrium && n_spins > 0) {
        BLOCH_CUDA(cudaMemcpyAsync(d_Mxy, h_Mxy, size_t(n_spins) * 2 * sizeof(float), cudaMemcpyHostToDevice, stream));
        BLOCH_CUDA(cudaMemcpyAsync(d_Mz, h_Mz, size_t(n_spins) * sizeof(float), cudaMemcpyHostToDevice, stream));
    }
    const size_t sig = signal_rows(plan, n_spins) * size_t(plan->info.n_adc) * sizeof(float2);
    float *d_v[3] = {nullptr, nullptr, nullptr};
    if (has_v) {
        const float *hv[3] = {h_vx, h_vy, h_vz};
        for (int k = 0; k < 3; ++k) {
            d_v[k] = (float *)(base + (10 + k) * arr);
            if (n_spins > 0)
                BLOCH_CUDA(cudaMemcpyAsync(d_v[k], hv[k], size_t(n_spins) * sizeof(float), cudaMemcpyHostToDevice, stream));
        }
    }
    float *d_sig = (float *)(base + 13 * arr);
    unsigned char *d_ws = base + 13 * arr + align_up(sig, kAlign);
    const size_t ws_bytes = scratch_bytes - (size_t)(d_ws - base);
    rc = bloch_simulate_motion(plan, n_spins, d[0], d[1], d[2], d[3], d[4], d[5], d[6], d_v[0], d_v[1], d_v[2], d_Mxy,
                               d_Mz, init_equilibrium, d_sig, d_ws, ws_bytes, stream_);
    if (rc) return rc;
    if (sig > 0) BLOCH_CUDA(cudaMemcpyAsync(h_signal, d_sig, sig, cudaMemcpyDeviceToHost, stream));
    if (h_Mxy && n_spins > 0) {
        BLOCH_CUDA(cudaMemcpyAsync(h_Mxy, d_Mxy, size_t(n_spins) * 2 * sizeof(float), cudaMemcpyDeviceToHost, stream));
        BLOCH_CUDA(cudaMemcpyAsync(h_Mz, d_Mz, size_t(n_spins) * sizeof(float), cudaMemcpyDeviceToHost, stream));
    }
    BLOCH_CUDA(cudaStreamSynchronize(stream));
    return collect_status(plan, nullptr);  // bad T1 / T2, non-finite input, phase range: see bloch_plan_status
}

int bloch_simulate_host_coils_scratch_bytes(const bloch_plan *plan, int64_t n_spins, int n_coils, size_t *out) {
    if (!plan || !out || n_spins < 0 || n_coils < 1) return fail(BLOCH_EINVAL, "NULL plan/out, negative n_spins or n_coils < 1");
    size_t ws = 0;
    int rc = bloch_plan_workspace_bytes_coils(plan, n_spins, n_coils, &ws);
    if (rc) return rc;
    const size_t arr = align_up(size_t(n_spins) * sizeof(float), kAlign);
    const size_t coil = align_up(size_t(n_coils) * size_t(n_spins) * sizeof(float2), kAlign);
    const size_t sig = align_up(size_t(n_coils) * size_t(plan->info.n_adc) * sizeof(float2), kAlign);
    *out = 13 * arr + coil + sig + ws + kAlign;
    return BLOCH_OK;
}

int bloch_simulate_host_coils(const bloch_plan *plan, int64_t n_spins, const float *h_x, const float *h_y,
                              const float *h_z, const float *h_M0, const float *h_T1, const float *h_T2,
                              const float *h_dw, int n_coils, const float *h_coil, float *h_Mxy, float *h_Mz,
                              int init_equilibrium, float *h_signal, void *d_scratch, size_t scratch_bytes,
                              void *stream_) {
    return bloch_simulate_host_coils_motion(plan, n_spins, h_x, h_y, h_z, h_M0, h_T1, h_T2, h_dw, nullptr, nullptr, nullptr,
                                            n_coils, h_coil, h_Mxy, h_Mz, init_equilibrium, h_signal, d_scratch,
                                            scratch_bytes, stream_);
}

int bloch_simulate_host_coils_motion(const bloch_plan *plan, int64_t n_spins, const float *h_x, const float *h_y,
                                     const float *h_z, const float *h_M0, const float *h_T1, const float *h_T2,
                                     const float *h_dw, const float *h_vx, const float *h_vy, const float *h_vz,
                                     int n_coils, const float *h_coil, float *h_Mxy, float *h_Mz, int init_equilibrium,
                                     float *h_signal, void *d_scratch, size_t scratch_bytes, void *stream_) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    const bool has_v = h_vx || h_vy || h_vz;
    if (has_v && !(h_vx && h_vy && h_vz)) return fail(BLOCH_EINVAL, "give all of h_vx, h_vy, h_vz or none");
    size_t need = 0;
    int rc = bloch_simulate_host_coils_scratch_bytes(plan, n_spins, n_coils, &need);
    if (rc) return rc;
    if (!d_scratch || scratch_bytes < need || (reinterpret_cast<uintptr_t>(d_scratch) % kAlign) != 0)
        return fail(BLOCH_EWORKSPACE, "scratch NULL, too small or not 256-B aligned");
    if (n_spins > 0 && (!h_x || !h_y || !h_z || !h_M0 || !h_T1 || !h_T2 || !h_dw || !h_coil))
        return fail(BLOCH_EINVAL, "NULL phantom or coil array");
    if (!init_equilibrium && (!h_Mxy || !h_Mz)) return fail(BLOCH_EINVAL, "initial state requested but h_Mxy/h_Mz NULL");
    if ((h_Mxy == nullptr) != (h_Mz == nullptr)) return fail(BLOCH_EINVAL, "h_Mxy and h_Mz must both be given or both NULL");
    if (plan->info.n_adc > 0 && !h_signal) return fail(BLOCH_EINVAL, "h_signal is NULL");
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t arr = align_up(size_t(n_spins) * sizeof(float), kAlign);
    const size_t coil = align_up(size_t(n_coils) * size_t(n_spins) * sizeof(float2), kAlign);
    const size_t sig = size_t(n_coils) * size_t(plan->info.n_adc) * sizeof(float2);
    unsigned char *base = (unsigned char *)d_scratch;
    float *d[7];
    const float *h[7] = {h_x, h_y, h_z, h_M0, h_T1, h_T2, h_dw};
    for (int k = 0; k < 7; ++k) {
        d[k] = (float *)(base + k * arr);
        if (n_spins > 0)
            BLOCH_CUDA(cudaMemcpyAsync(d[k], h[k], size_t(n_spins) * sizeof(float), cudaMemcpyHostToDevice, stream));
    }
    float *d_Mxy = h_Mxy ? (float *)(base + 7 * arr) : nullptr;
    float *d_Mz = h_Mz ? (float *)(base + 9 * arr) : nullptr;
    if (!init_equilibrium && n_spins > 0) {
        BLOCH_CUDA(cudaMemcpyAsync(d_Mxy, h_Mxy, size_t(n_spins) * 2 * sizeof(float), cudaMemcpyHostToDevice, stream));
        BLOCH_CUDA(cudaMemcpyAsync(d_Mz, h_Mz, size_t(n_spins) * sizeof(float), cudaMemcpyHostToDevice, stream));
    }
    float *d_v[3] = {nullptr, nullptr, nullptr};
    if (has_v) {
        const float *hv[3] = {h_vx, h_vy, h_vz};
        for (int k = 0; k < 3; ++k) {
            d_v[k] = (float *)(base + (10 + k) * arr);
            if (n_spins > 0)
                BLOCH_CUDA(cudaMemcpyAsync(d_v[k], hv[k], size_t(n_spins) * sizeof(float), cudaMemcpyHostToDevice, stream));
        }
    }
    float *d_coil = (float *)(base + 13 * arr);
    if (n_spins > 0)
        BLOCH_CUDA(cudaMemcpyAsync(d_coil, h_coil, size_t(n_coils) * size_t(n_spins) * sizeof(float2),
                                   cudaMemcpyHostToDevice, stream));
    float *d_sig = (float *)(base + 13 * arr + coil);
    unsigned char *d_ws = base + 13 * arr + coil + align_up(sig, kAlign);
    const size_t ws_bytes = scratch_bytes - (size_t)(d_ws - base);
    rc = bloch_simulate_coils_motion(plan, n_spins, d[0], d[1], d[2], d[3], d[4], d[5], d[6], d_v[0], d_v[1], d_v[2],
                                     n_coils, d_coil, d_Mxy, d_Mz, init_equilibrium, d_sig, d_ws, ws_bytes, stream_);
    if (rc) return rc;
    if (sig > 0) BLOCH_CUDA(cudaMemcpyAsync(h_signal, d_sig, sig, cudaMemcpyDeviceToHost, stream));
    if (h_Mxy && n_spins > 0) {
        BLOCH_CUDA(cudaMemcpyAsync(h_Mxy, d_Mxy, size_t(n_spins) * 2 * sizeof(float), cudaMemcpyDeviceToHost, stream));
        BLOCH_CUDA(cudaMemcpyAsync(h_Mz, d_Mz, size_t(n_spins) * sizeof(float), cudaMemcpyDeviceToHost, stream));
    }
    BLOCH_CUDA(cudaStreamSynchronize(stream));
    return collect_status(plan, nullptr);  // bad T1 / T2, non-finite input, phase range: see bloch_plan_status
}

// ---- bloch_simulate_static: the simulation with the library's OWN scratch memory, no allocation anywhere ----
// The workspace of bloch_simulate (packed spin records, the per-chunk partial signal rows signal_kernel / seq_kernel
// write and reduce_kernel sums, tickets) lives in this file-scope device array instead of a caller buffer.  Every
// context that loads the library holds these BLOCH_STATIC_WORKSPACE_BYTES until exit.  In host code the array's name
// is only a stand-in: the device address comes from cudaGetSymbolAddress, once per device with that device current.
static __device__ __align__(256) unsigned char g_static_workspace[BLOCH_STATIC_WORKSPACE_BYTES];

namespace bloch {
namespace {
std::atomic<void *> g_static_workspace_ptr[kMaxDevices];  // per device: the array's address in that device's context

// the current device's address of g_static_workspace (no allocation: the array is part of the loaded module)
int static_workspace(void **out) {
    int dev = 0;
    BLOCH_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(BLOCH_ECUDA, "device ordinal beyond the library's per-device table");
    void *p = g_static_workspace_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        BLOCH_CUDA(cudaGetSymbolAddress(&p, g_static_workspace));
        if (!p || (reinterpret_cast<uintptr_t>(p) % kAlign) != 0)
            return fail(BLOCH_ECUDA, "cudaGetSymbolAddress returned a NULL or misaligned static workspace");
        g_static_workspace_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return BLOCH_OK;
}
}  // namespace
}  // namespace bloch

int bloch_simulate_static(const bloch_plan *plan, int64_t n_spins, const float *d_x, const float *d_y,
                          const float *d_z, const float *d_M0, const float *d_T1, const float *d_T2,
                          const float *d_dw, float *d_Mxy, float *d_Mz, int init_equilibrium, float *d_signal,
                          void *stream_) {
    if (!plan) return fail(BLOCH_EINVAL, "NULL plan");
    if (n_spins < 0 || n_spins > INT32_MAX) return fail(BLOCH_EINVAL, "n_spins out of range");
    if (plan->info.motion_mode != BLOCH_MOTION_NONE)
        return fail(BLOCH_EINVAL, "bloch_simulate_static: static plans only (no motion); use bloch_simulate_motion");
    // the timing taps create CUDA events on first use: an allocation this entry point promises not to make
    if (plan->profiling)
        return fail(BLOCH_EINVAL, "bloch_simulate_static: switch bloch_plan_set_profiling off (its taps create CUDA events)");
    size_t need = 0;
    int rc = bloch_plan_workspace_bytes(plan, n_spins, &need);
    if (rc != BLOCH_OK) return rc;
    if (need > size_t(BLOCH_STATIC_WORKSPACE_BYTES)) {
        char msg[200];
        std::snprintf(msg, sizeof msg,
                      "bloch_simulate_static: %lld spins of this plan need %zu B of workspace, the static array holds %zu B; "
                      "use bloch_simulate with a caller workspace", (long long)n_spins, need, size_t(BLOCH_STATIC_WORKSPACE_BYTES));
        return fail(BLOCH_EWORKSPACE, msg);
    }
    void *ws = nullptr;
    if (n_spins > 0 && (rc = bloch::static_workspace(&ws)) != BLOCH_OK) return rc;
    // simulate_impl treats its workspace as uninitialised memory: it clears the findings word and the tickets of the
    // whole-sequence kernel on `stream` before the kernels that use them and overwrites everything else before
    // reading it, so the contents the previous call left in the array do not matter.
    return bloch::simulate_impl(plan, n_spins, d_x, d_y, d_z, d_M0, d_T1, d_T2, d_dw, nullptr, nullptr, nullptr, 0, nullptr,
                                d_Mxy, d_Mz, init_equilibrium, d_signal, ws, size_t(BLOCH_STATIC_WORKSPACE_BYTES), stream_);
}

int bloch_microbench(int kind, int iters, double *ops_per_s, void *stream_) {
    if (!ops_per_s || iters <= 0 || kind < 0 || kind > 3) return fail(BLOCH_EINVAL, "bad microbench argument");
    int rc = check_arch();
    if (rc) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    const int sms = sm_count_cached();
    const int grid = sms * 8, threads = 256;
    float *d_out = nullptr;
    BLOCH_CUDA(cudaMalloc(&d_out, sizeof(float)));  // diagnostic entry point only; not on the hot path
    cudaEvent_t e0, e1;
    BLOCH_CUDA(cudaEventCreate(&e0));
    BLOCH_CUDA(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        BLOCH_CUDA(cudaEventRecord(e0, stream));
        if (kind == 0) mb_mufu<<<grid, threads, 0, stream>>>(iters, d_out);
        else if (kind == 1) mb_ffma<<<grid, threads, 0, stream>>>(iters, d_out);
        else if (kind == 2) mb_dfma<<<grid, threads, 0, stream>>>(iters, d_out);
        else mb_ffma3<<<grid, threads, 0, stream>>>(iters, d_out);
        BLOCH_CUDA(cudaEventRecord(e1, stream));
        BLOCH_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        BLOCH_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    const double per_thread = kind == 0 ? 24.0 * iters : 32.0 * iters;
    *ops_per_s = per_thread * (double)grid * threads / (best * 1e-3);
    return BLOCH_OK;
}

}  // extern "C"
