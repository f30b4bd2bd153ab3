// awg_plan.h -- host-side plan state (shared by awg_plan.cu and awg_ring.cu).  CUDA path only.
#pragma once
#include <cstdint>
#include <utility>
#include <vector>

#include <cuda_runtime.h>

#include "awg.h"
#include "awg_internal.h"

namespace awg {

constexpr int kTableVersions = 4;  // device copies of the trajectory table in flight (updates never stall a running kernel)

// Current segment of one tone, host precision (x87 long double + 64-bit fixed-point turns).
struct HostTone {
    long double f0 = 0, f1 = 0;  // Hz: frequency before / after the current move
    long double T = 0;           // move duration, s
    long double Tn = 0;          // move duration, samples (T*fs)
    long double DT = 0;          // (f1-f0)*T, cycles
    long double expL = 0;        // AWG_PROFILE_EXP: ln(f1/f0); the phase gained over the carrier is f0 T (expm1(L s)/L - s)
    int64_t ns_int = 0;          // move start, samples: floor and
    double ns_frac = 0;          //   fractional part
    uint64_t theta_pre = 0, w_pre = 0;    // carrier before/during the move: turns*2^64, turns/sample*2^64
    uint64_t theta_post = 0, w_post = 0;  // carrier after the move
    float A = 0;
    int32_t profile = AWG_PROFILE_STATIC;
    int32_t cls = 0;
    // amplitude ramp (Eq. 9's a_j[i]): A -> A1 over [amp_ns, amp_ns + amp_Tn) samples along amp_prof
    float A1 = 0;
    int32_t amp_prof = AWG_PROFILE_STATIC;
    long double amp_ns = 0, amp_Tn = 0;
};

awg_status fail(awg_status code, const char *fmt, ...);
awg_status fail_cuda(cudaError_t e, const char *what);

}  // namespace awg

constexpr int kUseSlots = 4;   // streams tracked per table version (more: the oldest slot changes hands after a wait)
constexpr int kE2eSlots = 4;   // device staging slots of awg_synthesize_range_host

struct awg_plan {
    int32_t n_tones = 0, n_pad = 0;
    long double fs = 0;
    int64_t chunk_len = 0;
    double scale = 0;
    int32_t engine = AWG_ENGINE_MUFU;
    int device = 0;
    bool have_table = false;
    bool dirty_all = false;                 // whole table changed (awg_set_trajectories)
    std::vector<int32_t> dirty_tones;       // tones changed by updates since the last upload
    int64_t last_update_chunk = 0;
    std::vector<awg::HostTone> tones;
    // static-buffer pathway: tones served by the looped buffer X_static are not in the
    // device table; slot_of[k] is tone k's record in the device table, or -1
    std::vector<uint8_t> in_buffer;
    std::vector<int32_t> slot_of;
    int32_t n_active = 0;
    bool slow2 = false;               // some active tone carries CLS_SLOW2_FLAG (slow pass with two table corrections per thread)
    awg::FixGrid fix{};                 // fixed-point grids of the kernel's leaf merge for the current table (fix_grids())
    float *xs[2] = {};                      // X_static, chunk_len floats each; xs[xs_cur] is current (a fold writes the other)
    int xs_cur = 0;
    bool xs_on = false;
    unsigned char *dev_aux = nullptr;       // table of the tones whose period is being added to X_static
    unsigned char *dev_aux_stage = nullptr;
    unsigned char *host_aux = nullptr;      // pinned staging of their cores
    // versioned device tables
    size_t table_bytes = 0;
    int cur_version = 0;
    unsigned char *dev_table[awg::kTableVersions] = {};
    size_t core_bytes = 0;                                 // n_pad tone cores (what the host uploads)
    unsigned char *host_table[awg::kTableVersions] = {};  // pinned staging: tone cores, then int32 indices
    unsigned char *dev_stage[awg::kTableVersions] = {};   // device staging of the same layout (input of the expand kernel)
    // readers of each table version: one event per stream that has launched work on it (a plan is used from several
    // streams: the caller's, the two synthesis streams of awg_synthesize_range_host, the side streams of the multiplexer)
    struct VersionUse {
        cudaStream_t stream[kUseSlots] = {};
        cudaEvent_t ev[kUseSlots] = {};
        int n = 0;
    } use[awg::kTableVersions];
    cudaEvent_t uploaded[awg::kTableVersions] = {};
    cudaStream_t upload_stream[awg::kTableVersions] = {};
    // awg_synthesize_range_host
    int16_t *e2e_slot[kE2eSlots] = {};
    cudaStream_t e2e_stream[3] = {};        // two synthesis streams (alternating pieces), one copy stream
    cudaEvent_t e2e_ready[kE2eSlots] = {}, e2e_done[kE2eSlots] = {};
    std::vector<std::pair<int64_t, int64_t>> hot_tiles;   // (absolute tile, tones) where many slow movers start or end a move at once
    bool hot_dirty = true;                  //   (listed again after a table change)
    std::vector<int64_t> hot_scratch[2];
    bool e2e_ok = false;
    // awg_synthesize_chunk_mux, held by the plan of channel 0: channels 1.. run on these streams beside channel 0
    cudaStream_t mux_stream[7] = {};
    cudaEvent_t mux_fork = nullptr, mux_join[7] = {};
    int mux_n = 0;                          // streams and join events created so far                    // all slots, streams and events exist
    // accounting
    int64_t h2d_bytes = 0, d2h_bytes = 0;
    int n_rings = 0;
};

namespace awg {
awg_status ensure_table(awg_plan *p, cudaStream_t stream);
awg_status synthesize_samples(awg_plan *p, int64_t n_begin, int64_t n_count, void *dev_out, bool f32, cudaStream_t stream,
                              int32_t out_stride = 1, int32_t out_offset = 0);
awg_status check_chunk_call(awg_plan *p, int64_t first_chunk, int64_t n_chunks, const void *out, size_t align);
awg_status apply_update(awg_plan *p, int64_t chunk_idx, int32_t n_upd, const int32_t *tone_idx, const double *f1,
                        const double *t_dur, const int32_t *profile);
}  // namespace awg
