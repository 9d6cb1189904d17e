// internal.h -- plan representation shared by the host planner (plan.cpp) and the launcher (api.cu).
// Not part of the C ABI.  Nothing here is shared with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/bloch.h"

namespace bloch {

constexpr int kBlockPrecession = 0;
constexpr int kBlockRF = 1;
constexpr double kTimeTol = 1e-12;       // reading G13
constexpr int64_t kDefaultMaxBlockPoints = int64_t(1) << 22;
constexpr size_t kAlign = 256;
// device scalars written by pack_kernel (Workspace::scal) and mirrored to bloch_plan::h_status: all maxima are float
// bit patterns of non-negative values under an integer atomicMax (order-independent), the flags an atomicOr
constexpr int kScalR2Max = 0;    // max 1/T2
constexpr int kScalX2Max = 1;    // max x^2 + y^2 + z^2
constexpr int kScalDwMax = 2;    // max |dw|
constexpr int kScalV2Max = 3;    // max |v|^2
constexpr int kScalFlags = 4;    // BLOCH_STATUS_BAD_RELAXATION | BLOCH_STATUS_NONFINITE
constexpr int kScalValid = 5;    // 1 once pack_kernel has run (the host clears it when it has evaluated the findings)
constexpr int kStatusWords = 8;
constexpr double kFp32TurnLimit = 256.0;      // AUTO: fp32 phase up to here
constexpr double kFp64TurnLimit = 524288.0;   // 2^19: the fixed-point fraction of the fp64 phase (signal.cuh)

// RF block table (a4), read by rf_kernel through 1-D bulk copies (TMA) tile by tile:
//   [directory: n_tiles x {int32 byte offset from the block's table start, int32 bytes}, padded to 16 B]
//   [tile 0][tile 1]...      tile = RfTileHdr (64 B) + n_steps records, 16-B aligned
// A tile never mixes two step lengths dt (the planner cuts tiles where dt changes), so the relaxation
// factors of Eq 11 are per-tile constants of a spin.  Records:
//   compact (kRfFlagUniformG: gamma*dt*G identical for all steps of the tile, e.g. a slice-select plateau)
//       16 B  (wx, wy, wx^2 + wy^2, 0)          wx + i wy = gamma * dt * B1 (Eq 8)
//   general
//       32 B  (wx, wy, wx^2 + wy^2, 0) (gx, gy, gz, 0)      g = gamma * dt * mean G of the step (reading G5)
constexpr int kRfTileSteps = 128;
constexpr int kRfHdrBytes = 64;
//   motion (kRfFlagMotion, never compact)
//       48 B  general record + (hx, hy, hz, 0)     h = gamma * dt * (G_n t_n + G_{n+1} t_{n+1}) / 2, so that
//                                                  gamma Bz dt = g . x + h . v + dw dt for x(t) = x + v t
constexpr int kRfTileBytesMax = kRfHdrBytes + kRfTileSteps * 48;
constexpr int kRfFlagUniformG = 1;
constexpr int kRfFlagMotion = 2;
struct RfTileHdr {
    float wxy2_max, gx_max, gy_max, gz_max;  // max over the tile's steps of wx^2+wy^2, |gx|, |gy|, |gz|
    float dt;                                // step length [s], the same for every step of the tile
    int32_t n_steps;
    int32_t flags;
    float pad0;
    float gx, gy, gz, pad1;                  // the tile's gradient part when kRfFlagUniformG
    float hx_max, hy_max, hz_max, pad2;      // max |hx|, |hy|, |hz| (kRfFlagMotion)
};
static_assert(sizeof(RfTileHdr) == kRfHdrBytes, "RfTileHdr must be 64 B");

// A run of compact (uniform-gradient) RF tiles passed to rf_const_kernel BY VALUE as a kernel parameter: the step
// records then sit in the constant bank and reach the FMAs as uniform operands (no shared-memory staging, no barrier,
// fewer register-file reads per step).  <= 32,764 B of parameters per launch: 2000 steps of 16 B + 24 tile headers = 32,592 B.
constexpr int kRfConstSteps = 2000;
constexpr int kRfConstTiles = 24;
struct RfConstTile {
    int32_t n_steps;
    float dt, gx, gy, gz, wxy2_max;  // as RfTileHdr (uniform-gradient tiles: g*_max = |g*|)
};
struct RfConstArgs {
    int32_t n_tiles, n_steps, pad0, pad1;
    RfConstTile tile[kRfConstTiles];
    float rec[kRfConstSteps * 4];    // (wx, wy, wx^2 + wy^2, 0) per step, tile after tile: the 16-byte compact records
};
static_assert(sizeof(RfConstArgs) <= 32764 - 160, "kernel parameter budget: 32,764 B with the other arguments");

// One block of the time axis: a maximal run of RF-active intervals (excitation regime) or
// a run of RF-free intervals (precession regime), :132.
struct Block {
    int type = kBlockPrecession;
    int64_t first = 0;        // first interval
    int64_t count = 0;        // number of intervals
    int64_t adc_first = 0;    // precession: first ADC sample served, in ADC order
    int64_t adc_count = 0;    //             number of ADC samples served (= evaluated points of the signal kernel)
    int64_t table_off = 0;    // byte offset of this block's records in the table buffer
    int64_t lin_pts = 0;      // precession: leading samples (a multiple of 16) that signal_lin_kernel may serve, see plan.cpp
    int64_t n_tiles = 0;      // RF: tiles in the block's table (see RfTileHdr)
    int64_t rf_const_first = 0, rf_const_count = 0;  // RF: its chunks in bloch_plan::rf_const (0: not served by rf_const_kernel)
    // precession block end record: k' = -gamma_bar * K(T) [turns/m] and tau = T [s] (Eq 12-13)
    double kend[3] = {0, 0, 0};
    double tau_end = 0;
    double mend[3] = {0, 0, 0};  // motion: first moment mu' = -gamma_bar * sum (G_n t_n + G_{n+1} t_{n+1}) dt / 2 [turns s/m]
};

// Whole-sequence program for the fused kernel (seq.cuh): one 64-B descriptor per block, in block order, appended
// to the table buffer at bloch_plan::prog_off.
struct SeqOp {
    int32_t type;       // kBlockRF / kBlockPrecession
    int32_t n;          // RF: tiles of the block's table; precession: ADC samples served (evaluated points)
    int64_t table_off;  // byte offset of the block's records in the table buffer
    int64_t adc_first;  // precession: first ADC sample served, in ADC order
    int64_t pad;
    double kend[3];     // precession block end record: k' = -gamma_bar K(T) [turns/m]   (offset 32: read as double4)
    double tau_end;     //                              T [s]
};
static_assert(sizeof(SeqOp) == 64, "SeqOp must be 64 B");

// The largest launch of each kernel kind in the last simulation (bloch_plan_last_kernel): what a profiler capture of
// "the dominant kernel" must match to describe this binary and this workload.
struct KernelNote {
    char name[56] = {0};  // as ncu prints it, e.g. "rf_kernel<0>", "signal_kernel<8, 0, 0>"
    int64_t grid = 0;     // CTAs
    int block = 0;        // threads per CTA
};

// The ADC-bearing precession blocks in order (appended to the table buffer at bloch_plan::adcblk_off): what the fused
// kernel's lagging sum over CTAs needs to know about a block it finished a few blocks ago.
struct SeqAdcBlock {
    int64_t adc_first;
    int32_t n;
    int32_t pad;
};
static_assert(sizeof(SeqAdcBlock) == 16, "SeqAdcBlock must be 16 B");

struct Timing {
    float ms_rf = 0, ms_prec = 0, ms_total = 0;
    int64_t launches = 0;
};

}  // namespace bloch

struct bloch_plan {
    double gamma = 0;
    bloch_sim_params params{};
    bloch_plan_info info{};
    std::vector<bloch::Block> blocks;
    std::vector<unsigned char> tables;   // host staging copy of the device tables
    std::vector<bloch::RfConstArgs> rf_const;   // static plans: the compact RF tiles again, as kernel-parameter blocks (rf_const_kernel)
    const unsigned char *d_tables = nullptr;
    int64_t prog_off = 0;                // byte offset of the SeqOp program in the table buffer
    int64_t n_adc_blocks = 0;            // precession blocks that serve ADC samples
    int64_t adcblk_off = 0;              // byte offset of the SeqAdcBlock array in the table buffer
    int path = 0;                        // BLOCH_PATH_*
    int opt[BLOCH_N_OPTIONS] = {1, 0, 0, 4, 0, 0, -1, -1, -1, 0, 1};  // BLOCH_OPT_* defaults (bloch_plan_set_option)
    // phase-range bookkeeping (bloch_sim_params extents): largest |k'| [turns/m], tau [s] and |mu'| [turns s/m] of
    // any evaluated point (block ends included), and the largest phase within the declared extents
    double k_max = 0, tau_max = 0, m_max = 0, worst_turns = 0;
    double ext_m = 0.25, ext_hz = 1000.0, ext_mps = 1.0;
    int phase_requested = 0;
    // findings of the last simulation's pack_kernel (kStatusWords words), copied here by the simulation itself;
    // pinned host memory, allocated by bloch_plan_upload
    unsigned *h_status = nullptr;
    // profiling taps
    bool profiling = false;
    mutable std::vector<void *> events;  // cudaEvent_t pool
    mutable std::vector<int> event_kind; // per interval between events: 0 other, 1 rf, 2 precession
    mutable bloch::Timing last{};
    mutable bloch::KernelNote last_kernel[BLOCH_N_KINDS];
};

namespace bloch {
void set_error(const std::string &msg);
int fail(int code, const std::string &msg);
int build_plan(const bloch_scanner *scanner, const bloch_sequence *seq, const bloch_sim_params *params,
               bloch_plan *plan);
}  // namespace bloch
