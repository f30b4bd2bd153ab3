// awg_internal.h -- types shared by the host side (plan / trajectory table) and the kernels.
// CUDA path only: nothing under oracle/ includes this.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "awg.h"

namespace awg {

// Tone classes: how the in-tile phase polynomial of a MOVING tile is evaluated (hot-path step a2).
// Chosen per tone on the host from worst-case bounds on the dropped Taylor terms.
enum : int32_t {
    CLS_STATIC = 0,  // never moves (profile STATIC or f1 == f0): carrier only
    CLS_QUAD = 2,    // moving tiles need the k^2 term only (LINEAR always; slow MINJERK)
    CLS_DEG4 = 4,    // k^2..k^4
    CLS_DEG6 = 6,    // k^2..k^6 (exact Taylor series of the degree-6 min-jerk phase)
    CLS_EXACT = 7    // fp32 in-tile polynomial not accurate enough: moving tiles use the fp64 path
};

// Device trajectory table, structure of arrays (hot-path step a0).  Phases are in TURNS as unsigned
// 64-bit fixed point (1 turn = 2^64), so carrier phase theta + w*n wraps exactly mod 1 for any n:
// this is the range reduction of Eq. 14 done in integer arithmetic.
//   before the move   (u <= 0):      phase = theta_pre  + w_pre *n
//   during the move (0 < u < Tn):    phase = theta_pre  + w_pre *n + DT*g(u/Tn)     g = s^2/2 or 5/2 s^4 - 3 s^5 + s^6
//   after the move    (u >= Tn):     phase = theta_post + w_post*n
// with u = (n - ns_int) - ns_frac the (real) number of samples since the move started.
struct ToneTable {
    const uint64_t *theta_pre;   // [N]
    const uint64_t *w_pre;       // [N] frac(f0/fs) * 2^64
    const uint64_t *theta_post;  // [N]
    const uint64_t *w_post;      // [N] frac(f1/fs) * 2^64
    const int64_t *ns_int;       // [N] floor(t_start*fs)
    const double *ns_frac;       // [N] t_start*fs - ns_int, in [0,1)
    const double *Tn;            // [N] t_dur*fs (samples, real)
    const double *inv_Tn;        // [N]
    const double *DT;            // [N] (f1-f0)*t_dur, cycles
    const float *A;              // [N]
    const int32_t *cls;          // [N] (profile << 8) | CLS_*
    int32_t n_tones;
};

constexpr int kTableArrays64 = 9;  // the nine 8-byte arrays above, in this order
constexpr size_t table_bytes(int n_pad) { return size_t(n_pad) * (kTableArrays64 * 8 + 4 + 4); }

struct LaunchParams {
    ToneTable tab;
    int64_t n_begin;   // absolute index of the first output sample (multiple of 8)
    int64_t n_count;   // samples to produce (multiple of 8)
    float scale;       // int16 full-scale factor
    void *out;         // int16* or float* (device)
    int32_t out_f32;   // 0: int16 codes, 1: fp32 sum before quantisation
};

cudaError_t launch_mufu(const LaunchParams &lp, cudaStream_t stream);
cudaError_t launch_fp64(const LaunchParams &lp, cudaStream_t stream);
void count_launch();

}  // namespace awg
