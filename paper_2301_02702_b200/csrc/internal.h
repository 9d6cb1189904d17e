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
    const unsigned char *d_tables = nullptr;
    int64_t prog_off = 0;                // byte offset of the SeqOp program in the table buffer
    int path = 0;                        // BLOCH_PATH_*
    // profiling taps
    bool profiling = false;
    mutable std::vector<void *> events;  // cudaEvent_t pool
    mutable std::vector<int> event_kind; // per interval between events: 0 other, 1 rf, 2 precession
    mutable bloch::Timing last{};
};

namespace bloch {
void set_error(const std::string &msg);
int fail(int code, const std::string &msg);
int build_plan(const bloch_scanner *scanner, const bloch_sequence *seq, const bloch_sim_params *params,
               bloch_plan *plan);
}  // namespace bloch
