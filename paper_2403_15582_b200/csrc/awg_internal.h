// awg_internal.h -- types shared by the host side (plan / trajectory table) and the kernels.
// CUDA path only: nothing under oracle/ includes this.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "awg.h"

namespace awg {

// Tone classes: how the in-block phase polynomial of a MOVING block is evaluated (hot-path step a2).
// Chosen per tone on the host from worst-case bounds on the dropped Taylor terms.
enum : int32_t {
    CLS_STATIC = 0,  // never moves (profile STATIC or f1 == f0): carrier only
    CLS_QUAD = 2,    // moving blocks need the k^2 term only (LINEAR always; slow MINJERK)
    CLS_DEG4 = 4,    // k^2..k^4
    CLS_DEG6 = 6,    // k^2..k^6 (exact Taylor series of the degree-6 min-jerk phase)
    CLS_EXACT = 7,   // fp32 in-block polynomial not accurate enough: moving blocks use the fp64 path
    CLS_SLOW_FLAG = 1 << 16,  // OR-ed into ToneRec::cls: tiles wholly inside the move may take the slow pass (FMA pipe)
    CLS_SLOW2_FLAG = 1 << 18, // with CLS_SLOW_FLAG: the slow pass corrects the pair tables per PAIR of groups (two local frequencies per thread)
    CLS_AMP_FLAG = 1 << 17    // OR-ed into ToneRec::cls: the tone has an amplitude ramp (A -> A1 over [amp_ns, amp_ns + amp_Tn))
};

// Kernel geometry.  A thread owns kSPT consecutive samples of a block; a block is 32 lanes x kSPT = 512 samples
// (the span of one phase re-centring); a warp tile is kBlocksPerTile consecutive blocks, anchored at absolute
// sample indices that are multiples of kTile.
constexpr int kSPT = 16;
constexpr int kBlock = 32 * kSPT;
constexpr int kBlocksPerTile = 4;
constexpr int kTile = kBlocksPerTile * kBlock;
constexpr int kPairs = kSPT / 2;  // symmetric sample pairs per thread: centre +- (j + 1/2), j = 0..kPairs-1

// (the table of the pre-move carrier carries the amplitude A, the table of the post-move carrier A1: tiles after both
// the move and the ramp use the latter, tiles before both the former, anything in between takes the MUFU pass)
// Carrier table of the angle-addition engine (hot-path step a3, static tiles): with phi the carrier phase at the
// half-integer centre of a thread's 16 samples, the samples at centre +- (j + 1/2) are
//     A sin(phi +- (j+1/2) w) = sin(phi) * [A cos((j+1/2) w)]  +-  cos(phi) * [A sin((j+1/2) w)]
// so ONE multiply-add per tone-sample accumulates the even part P_j and the odd part Q_j.  Built on the device
// (awg_expand_kernel) from the 64-bit fixed-point frequency.
struct __align__(16) RotTable {
    float C[kPairs];    // A cos(2 pi (j + 1/2) w)
    float S[kPairs];    // A sin(2 pi (j + 1/2) w)
    float pad_[4];      // {cos, sin}(2 pi 32 w): rotation by two groups of 16 samples (static pass), 0, 0
};
static_assert(sizeof(RotTable) == 80, "RotTable must be 80 bytes");

// What the host uploads per tone (hot-path step a0): carriers, move window, move polynomial.  Phases are in TURNS as
// unsigned 64-bit fixed point (1 turn = 2^64), so the carrier phase theta + w*n wraps exactly mod 1 for any n: the
// range reduction of Eq. 14 done in integer arithmetic.  With u = (n - ns_int) - ns_frac the real
// number of samples since the move began:
//   before the move   (u <= 0):      phase = theta_pre  + w_pre *n
//   during the move (0 < u < Tn):    phase = theta_pre  + w_pre *n + DT*g(u/Tn)    g = s^2/2 or 5/2 s^4 - 3 s^5 + s^6
//   after the move    (u >= Tn):     phase = theta_post + w_post*n
struct __align__(16) ToneCore {
    // ---- 64 bytes: carriers and move window
    float A;               // amplitude
    int32_t cls;           // (profile << 8) | CLS_* [| CLS_SLOW_FLAG]
    uint64_t theta_pre;    // turns * 2^64
    uint64_t w_pre;        // frac(f0/fs) * 2^64
    uint64_t theta_post;
    uint64_t w_post;       // frac(f1/fs) * 2^64
    double ns_int;         // floor(t_start*fs), an exact integer (|.| < 2^53)
    double ns_frac;        // t_start*fs - ns_int, in [0,1)
    double Tn;             // t_dur*fs, samples (real)
    // ---- 64 bytes: move polynomial
    double inv_Tn;
    double DT;             // (f1-f0)*t_dur, cycles
    double q1;             // DT/Tn = (f1-f0)/fs, cycles per sample
    float q[5];            // q[k-2] = 2*pi*DT/Tn^k/k!, k = 2..6: radians per sample^k for unit g^(k)
                           // (AWG_PROFILE_EXP: q[0..3] hold f0*T in cycles and ln(f1/f0) as two doubles)
    // ---- amplitude ramp a_j[i] of Eq. 9: A before amp_ns, A + (A1 - A) h((n - amp_ns)/amp_Tn) during,
    // A1 after; h(s) = s or 10 s^3 - 15 s^4 + 6 s^5 (amp_prof).  A1 = A and amp_prof = STATIC without a ramp.
    float A1;
    double amp_ns;         // ramp start, samples (real)
    float amp_Tn;          // ramp duration, samples
    int32_t amp_prof;      // AWG_PROFILE_*
};
static_assert(sizeof(ToneCore) == 128, "ToneCore must be 128 bytes");

// Device trajectory table: one 288-byte record per tone (core + the tables of the two carriers), read by one lane per
// (tone, tile) with 16-byte loads.
struct __align__(16) ToneRec {
    ToneCore core;
    RotTable rot_pre;
    RotTable rot_post;
};
static_assert(sizeof(ToneRec) == 288, "ToneRec must be 288 bytes");

// Fixed-point grids on which the leaves of a large table are merged (exact integer sums; awg_kernels.cu).  A leaf's fp32
// sum v is first rounded to its OWN grid 2^-leaf_sh[leaf] (|v 2^leaf_sh| < 2^22: one fused multiply-add against 1.5 * 2^23)
// whose step follows the leaf's own sum of amplitudes, then shifted on to the common grid 2^-fix_sh on which no partial
// sum of the table reaches 2^30; quad_sh: the same for the summed moving tones of a quad.
struct FixGrid {
    int32_t fix_sh;
    float fix_inv;       // 2^-fix_sh
    int8_t leaf_sh[64];  // [quad * 4 + rank]
    int8_t quad_sh[16];
    uint32_t bias_q[16]; // bits(1.5 * 2^23) * sum over the quad's leaves of 2^(fix_sh - leaf_sh), mod 2^32: the magic-number bias parked with them
};

constexpr int kMaxHotTiles = 16;

struct LaunchParams {
    const ToneRec *tab;
    int32_t n_tones;
    int32_t out_f32;   // 0: int16 codes, 1: fp32 sum before quantisation
    int32_t slow2;     // != 0: some tone of the table carries CLS_SLOW2_FLAG: the slow pass corrects the pair tables per pair of groups
    int64_t n_begin;   // absolute index of the first output sample (multiple of 8)
    int64_t n_count;   // samples to produce (multiple of 8)
    float scale;       // int16 full-scale factor
    float qlo, qhi;    // clamp bounds of the quantiser in units of V (filled in by launch_synth)
    void *out;         // int16* or float* (device)
    int32_t out_stride;   // int16 output: code of sample n goes to out[(n - n_begin) * out_stride + out_offset]
    int32_t out_offset;   //   (channel multiplexing); fp32 output is always contiguous
    const float *xs;   // looped static buffer X_static (Eq. 9) added before quantisation, or nullptr
    int64_t xs_len;    //   its length L_s (a multiple of 8, >= kTile)
    uint32_t *sched;   // {next tile, teams finished}: the launch's tile-scheduler slot (filled in by launch_synth)
    // tone groups (tone_groups(); filled in by launch_synth): a team's warp takes `per` tones of quad q, a tile has n_quads quads
    int32_t per;
    int32_t n_quads;
    int32_t cross;       // != 0: the quads of a tile are separate work units (launches with few tiles); their sums meet in `scratch`
    int32_t *scratch;    //   [tile][block][kBlock] int32 fixed point, this launch's slot (zero before and after the launch)
    uint32_t *tile_cnt;  //   quads delivered per tile (zero before and after the launch)
    FixGrid fix;         // fixed-point grids of the leaf merge (fix_grids(); large tables only)
    // Tiles in which many tones start or end a move at once (all of them leave the angle-addition passes there) cost several
    // ordinary tiles; drawn late by the tile scheduler such a tile is the tail of the whole launch.  The host lists them
    // (ascending, relative to the launch's first tile) and the scheduler serves them first.  Which team computes a tile, and
    // when, has no effect on its samples.
    int32_t n_hot = 0;
    int32_t hot[kMaxHotTiles] = {};
};

// Warps of a team share a tile, each taking 1/split of the tones.  A function of the tone count ONLY, never of the
// launch size: the order in which tone partial sums are added is then the same for every chunking (bit-identical
// output across chunk sizes, include/awg.h "pure function").
int split_for(int n_tones);
// Tone groups of the synthesis kernel: `split` warps share a tile, warp `rank` takes `per` tones of each of the `quads`
// quads.  Functions of the tone count only (see split_for): the grouping fixes the fp32 summation order.
void tone_groups(int n_tones, int *split, int *per, int *quads);
// amp: max(|A|, |A1|) per tone of the table (host array, n_tones entries)
void fix_grids(const float *amp, int n_tones, FixGrid *out);

cudaError_t launch_synth(const LaunchParams &lp, int engine, cudaStream_t stream);
// table[idx ? idx[j] : j] = expand(src[j]) for j < n: copies the core and builds both carrier tables (fp64 sincospi)
cudaError_t launch_expand(ToneRec *table, const ToneCore *src, const int32_t *idx, int n, cudaStream_t stream);
void count_launch();

// ---- the allocation-free entry point (awg_synthesize_noalloc; include/awg.h) -----------------------------------------
constexpr int kNoAllocMaxTones = 4096;
constexpr int64_t kNoAllocMaxSamples = int64_t(1) << 20;
// cores: n_up = n_tones rounded up to 32 host tone cores (zero padded).  lp: tab, sched, tile_cnt, scratch, qlo, qhi and the
// tone groups are filled in here; everything the launch needs on the device lives in one static __device__ array.
cudaError_t launch_synth_noalloc(const ToneCore *cores, int n_up, const LaunchParams &lp, cudaStream_t stream);

}  // namespace awg
