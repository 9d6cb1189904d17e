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
constexpr int kRfStepFloats = 8;         // (wx, wy, gx, gy, gz, dt, 0, 0) per RF step

// One block of the time axis: a maximal run of RF-active intervals (excitation regime) or
// a run of RF-free intervals (precession regime), :132.
struct Block {
    int type = kBlockPrecession;
    int64_t first = 0;        // first interval
    int64_t count = 0;        // number of intervals
    int64_t adc_first = 0;    // precession: first ADC sample served, in ADC order
    int64_t adc_count = 0;    //             number of ADC samples served (= evaluated points of the signal kernel)
    int64_t table_off = 0;    // byte offset of this block's records in the table buffer
    // precession block end record: k' = -gamma_bar * K(T) [turns/m] and tau = T [s] (Eq 12-13)
    double kend[3] = {0, 0, 0};
    double tau_end = 0;
};

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
