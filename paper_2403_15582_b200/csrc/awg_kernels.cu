// awg_kernels.cu -- sm_100a synthesis kernels: the fused WG + WC (+ quantise) of PAPER.md:158-186.
//
// Hot-path steps (SURVEY.md section 8(a) / DESIGN.md section 6):
//   a1  re-centring in 64-bit fixed point + fp64: per (tone, 2048-sample tile) a u32 carrier for tones static there
//       (stage of the static pass in awg_synth_kernel), per (tone, 512-sample block) c0, c1, c2..c6 and the record
//       kind for tones moving there                                                          block_prologue()
//   a2  per tone-sample phase of a moving tone: c0 + c1*k (u32 turns, wraps exactly) + fp32 polynomial  mufu_rec<KIND>()
//   a3  sine.  Tiles in which a tone is static (angle-addition engine; a thread owns 64 consecutive samples, four groups of
//       16): per (thread, tone) two MUFU.SIN/COS pairs and a packed rotation give sin, cos at the pair centres of the four
//       groups, then per symmetric sample pair centre +- (j + 1/2)
//           A sin(phi +- (j+1/2) w) = sin(phi) [A cos((j+1/2) w)]  +-  cos(phi) [A sin((j+1/2) w)]
//       i.e. ONE fp32 multiply-add per tone-sample into the even/odd accumulators P_j, Q_j    sincos_tile(), pq_add()
//       Tiles wholly inside a SLOW move: a cubic phase polynomial gives the phase at the four pair centres, the pair tables
//       are moved to the thread's local frequency once (first order): 1.25 multiply-adds per tone-sample (1.5 with one
//       correction per pair of groups, SLOW2)                                     stage_slow(), slow_sincos(), slow_fma()
//       Blocks in which a tone moves otherwise (and every tone-sample of the MUFU engine): one MUFU.SIN each   mufu_rec<KIND>()
//   a4  fp32 register accumulation over tones: 4 groups x 16 samples per thread (angle-addition passes), 16 (MUFU pass);
//       tables above 256 tones: leaves of <= 64 (128) tones summed from zero, merged in int32 fixed point (exact), so that
//       launches with few tiles spread a tile's tones over CTAs bit-identically          ipark_leaf(), tone_groups(), fix_grids()
//   a5  quantise: round-half-even and saturate to int16 (fused multiply-add against 1.5*2^23)  pack8()
//   a6  two 16-byte stores of 8 consecutive int16 per thread and block                       store_block()
// No tensor cores (north_star), no per-tone wavetable in DRAM (the paper's limiter); output
// traffic is 2 bytes per sample.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <atomic>
#include <mutex>
#include <unordered_map>

#include "awg_internal.h"

namespace awg {

static std::atomic<int64_t> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

int split_for(int n_tones)
{
    // >= 5 tones per warp, at most one CTA (4 warps) per tile: a tile's latency is one warp's walk over its tones and over the
    // blocks it owns in the MUFU pass, and launches of a few dozen tones are bound by it (20 tones x 2^18 samples: 16.7 us with
    // one warp per tile, 8.5 us with four; 2^22 samples: 19.0 -> 20.7 us)
    int split = 1;
    while (split < 4 && n_tones / (split * 2) >= 5) split *= 2;
    return split;
}

void tone_groups(int n_tones, int *split, int *per, int *quads)
{
    const int sp = split_for(n_tones);
    int q = 1;
    // Large tables are cut into leaves of <= 64 tones (<= 128 above 2048 tones), four per quad, at most 16 quads: a leaf is
    // summed from zero in fp32 and the leaves are merged in fixed point (exact), so a launch with few tiles can spread a
    // tile's quads over CTAs and still produce the same bits as a large launch that walks them inside one CTA.  Measured
    // cost of the leaf boundaries in a large launch: 1 % (4096 tones, 8 quads) to 3 % (1000 tones, 4 quads).
    const int leaf = n_tones <= 2048 ? 64 : 128;
    if (sp == 4 && n_tones > 4 * leaf) {
        q = (n_tones + 4 * leaf - 1) / (4 * leaf);
        if (q > 16) q = 16;
    }
    int pr = (n_tones + sp * q - 1) / (sp * q);
    if (pr < 1) pr = 1;                        // (an empty table: every tone is served by the static buffer)
    q = (n_tones + sp * pr - 1) / (sp * pr);   // no empty quad
    if (q < 1) q = 1;
    *split = sp;
    *per = pr;
    *quads = q;
}

static int exponent_above(double a)
{
    // smallest e with a (1 + margin) < 2^e; sums of amplitudes down to 2^-64 keep their own grid
    int ex = 0;
    a = a * 1.001 + 5e-20;
    (void)std::frexp(a, &ex);   // a = m 2^ex, m in [1/2, 1)
    return ex;
}

void fix_grids(const float *amp, int n_tones, FixGrid *out)
{
    int split = 1, per = 1, quads = 1;
    tone_groups(n_tones, &split, &per, &quads);
    FixGrid g{};
    double total = 0.0;
    for (int t = 0; t < n_tones; ++t) total += static_cast<double>(amp[t]);
    g.fix_sh = 30 - exponent_above(total);
    g.fix_inv = static_cast<float>(std::ldexp(1.0, -g.fix_sh));
    for (int q = 0; q < 16; ++q) {
        double aq = 0.0;
        g.bias_q[q] = 0;
        for (int r = 0; r < 4; ++r) {
            double al = 0.0;
            if (q < quads && r < split) {
                const int t0 = std::min((q * split + r) * per, n_tones), t1 = std::min(n_tones, t0 + per);
                for (int t = t0; t < t1; ++t) al += static_cast<double>(amp[t]);
            }
            aq += al;
            g.leaf_sh[q * 4 + r] = static_cast<int8_t>(std::min(22 - exponent_above(al), g.fix_sh));
            if (q < quads && r < split) g.bias_q[q] += 0x4B400000u * (1u << (g.fix_sh - g.leaf_sh[q * 4 + r]));
        }
        g.quad_sh[q] = static_cast<int8_t>(std::min(22 - exponent_above(aq), g.fix_sh));
    }
    *out = g;
}

namespace {

constexpr int kHalf = kBlock / 2;     // Taylor expansions are centred on the block
constexpr int kWarps = 4;             // warps per CTA
constexpr int kCtasPerSm = 3;         // 12 warps per SM leave 168 registers per thread: tables and sines double-buffered
constexpr int kBatch = 32;            // tones (pass 1) or (tone, block) items (pass 2) per batch: one per lane
constexpr int kMaxBatches = 65536 / kWarps / kBatch;   // per warp (all its leaves), at the largest tone count and widest split
constexpr int kMaxQuads = 16;                          // leaves per warp and tile (awg::tone_groups)
constexpr float kTurnToRad = 1.4629180792671596e-9f;   // 2*pi / 2^32: int32 phase (turns * 2^32) -> radians
constexpr double kTwo64 = 18446744073709551616.0;
constexpr int kListBatches = 8;                        // batches of 32 tones compacted at a time for the MUFU pass
constexpr int kListCap = kListBatches * kBatch;
constexpr float kRoundMagic = 12582912.f;              // 1.5 * 2^23: fma(v, scale, magic) has the rounded integer in its low mantissa bits

__device__ __forceinline__ float mufu_sin(float x_rad)
{
    float y;
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x_rad));
    return y;
}

__device__ __forceinline__ float mufu_cos(float x_rad)
{
    float y;
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x_rad));
    return y;
}

__device__ __forceinline__ float2 dup2(float v) { return make_float2(v, v); }

__device__ __forceinline__ uint32_t round32(uint64_t turns64)
{
    return static_cast<uint32_t>((turns64 + 0x80000000ull) >> 32);
}

// frac(x) as 64-bit fixed-point turns; x in cycles, any sign, |x| < 2^52.
__device__ __forceinline__ uint64_t frac_to_fix64(double x)
{
    double fr = x - floor(x);
    return __double2ull_rz(fr * kTwo64);  // saturating at 2^64-1 when fr rounds to 1.0: error 2^-64 turn
}

__device__ __forceinline__ uint4 ldg16(const void *p) { return __ldg(reinterpret_cast<const uint4 *>(p)); }
__device__ __forceinline__ uint64_t u64_of(uint32_t lo, uint32_t hi) { return (static_cast<uint64_t>(hi) << 32) | lo; }
__device__ __forceinline__ double f64_of(uint32_t lo, uint32_t hi) { return __hiloint2double(static_cast<int>(hi), static_cast<int>(lo)); }

// g(s) of the move profile: phase gained over the carrier is DT*g(s) cycles.
__device__ __forceinline__ double profile_g(int profile, double s)
{
    if (profile == AWG_PROFILE_LINEAR) return 0.5 * s * s;
    double s2 = s * s;
    return s2 * s2 * (2.5 + s * (s - 3.0));  // 5/2 s^4 - 3 s^5 + s^6   (Eq. 10 p(i), prefactor T: G1)
}

// Exact (fp64 + 64-bit fixed point) phase of tone record r at absolute sample n, in turns * 2^64.
__device__ __forceinline__ uint64_t exact_phase(const ToneCore &r, int64_t n)
{
    if ((r.cls & 0xff) == CLS_STATIC) return r.theta_pre + r.w_pre * static_cast<uint64_t>(n);
    const double u = (static_cast<double>(n) - r.ns_int) - r.ns_frac;
    if (u <= 0.0) return r.theta_pre + r.w_pre * static_cast<uint64_t>(n);
    if (u >= r.Tn) return r.theta_post + r.w_post * static_cast<uint64_t>(n);
    const int profile = (r.cls >> 8) & 0xff;
    double x;
    if (profile == AWG_PROFILE_EXP) {
        // exponential chirp (G20): cycles gained over the carrier = f0 T (expm1(L s)/L - s), L = ln(f1/f0);
        // q[0..3] hold f0 T and L as two doubles
        const double F = *reinterpret_cast<const double *>(&r.q[0]), L = *reinterpret_cast<const double *>(&r.q[2]);
        const double s = u * r.inv_Tn;
        x = F * (expm1(L * s) / L - s);
    } else {
        x = r.DT * profile_g(profile, u * r.inv_Tn);
    }
    return r.theta_pre + r.w_pre * static_cast<uint64_t>(n) + frac_to_fix64(x);
}

// a_j[i] of Eq. 9 for a tone with an amplitude ramp, at absolute sample n.
__device__ __forceinline__ float amp_at(const ToneCore &r, int64_t n)
{
    if (!(r.cls & CLS_AMP_FLAG)) return r.A;
    const float u = static_cast<float>(static_cast<double>(n) - r.amp_ns);
    float s = r.amp_Tn > 0.f ? u / r.amp_Tn : (u >= 0.f ? 1.f : 0.f);
    s = fminf(fmaxf(s, 0.f), 1.f);
    const float h = r.amp_prof == AWG_PROFILE_LINEAR ? s : s * s * s * (10.f + s * (6.f * s - 15.f));
    return fmaf(r.A1 - r.A, h, r.A);
}

// Kinds of (tone, block) record, in the order the inner loops run them.
enum : int {
    K_NONE = -1,
    K_STATIC = 0,  // carrier only
    K_QUAD = 1,    // + k^2 term
    K_DEG4 = 2,    // + k^2..k^4
    K_DEG6 = 3,    // + k^2..k^6
    K_SBEG = 4,    // the move starts inside this block: pre-move carrier + P(max(k - kb, 0))
    K_SEND = 5,    // the move ends inside this block:  post-move carrier + P(max(kb - k, 0))
    K_EXACT = 6,   // anything else (both ends in one block, T = 0, CLS_EXACT tones): fp64 per sample
    K_XEDGE = 7,   // an exponential chirp starts or ends inside this block: carrier valid outside + P(max(+-(k - kb), 0))
    K_COUNT = 8
};

// One re-centred (tone, block) record:
//   phase(k) = c0 + c1*k [u32 turns, wrapping] + poly(k) [radians, fp32],  k = n - block centre
//   K_QUAD..K_DEG6: poly = k^2 (c2 + k (c3 + k (c4 + k (c5 + k c6))))     (Taylor series about the block centre)
//   K_SBEG/K_SEND:  poly = w^2 (c2 + w^2 (c3 + w (c4 + w c5))), w = max(+-(k - kb), 0), c6 = +-kb
//   K_XEDGE:        poly = w^2 (c2 + w (c3 + w c4)), w = max(c5 k - c6, 0), c5 = +-1, c6 = +-kb
struct BlockRec {
    uint32_t c0, c1;
    float A;
    float c2, c3, c4, c5, c6;
    int kind;
};

// Exponential chirp f0 e^(L s), s = u/Tn (G20): the (tone, block) record of a tone of that profile (class below
// CLS_EXACT).  Kept out of line and self-contained (it loads the core itself): the fp64 exponentials are needed for these
// tones only and must weigh neither on the registers nor on the schedule of block_prologue().
// q[0..3] of the core hold F = f0 T (cycles) and L = ln(f1/f0) as doubles; nc = the block's centre, bb_d = its first sample.
struct ExpRec {
    uint32_t c0, c1;
    float c2, c3, c4, c5, c6;
    int kind;
};
__device__ __noinline__ ExpRec exp_block(const ToneRec *rec, int c, uint64_t nc, double bb_d)
{
    const ToneCore &t = rec->core;
    ExpRec r;
    r.c2 = r.c3 = r.c4 = r.c5 = r.c6 = 0.f;
    r.kind = K_STATIC;
    const double ua = (bb_d - t.ns_int) - t.ns_frac;   // u of the block's first sample
    const double ub = ua + static_cast<double>(kBlock - 1);
    const double Tn = t.Tn, rT = t.inv_Tn;
    uint64_t ph, w;
    if (ub <= 0.0) {
        w = t.w_pre;
        ph = t.theta_pre + w * nc;
    } else if (ua >= Tn) {
        w = t.w_post;
        ph = t.theta_post + w * nc;
    } else if (ua < 0.0 && ub > Tn) {
        r.kind = K_EXACT;   // (the caller stores the tone index)
        r.c0 = r.c1 = 0;
        return r;
    } else {
        const double F = *reinterpret_cast<const double *>(&t.q[0]), L = *reinterpret_cast<const double *>(&t.q[2]);
        const double f0s = F * rT;   // f0/fs, cycles per sample
        if (ua < 0.0 || ub > Tn) {
            // One end of the move inside the block.  With w the (clamped) distance into the move from that end the phase
            // over the carrier valid outside is a power series that starts at w^2:
            //   start: f0/fs sum_k a^(k-1) w^k / k!     end: -f1/fs sum_k (-a)^(k-1) w^k / k!     (k >= 2; cycles; a = L/Tn)
            // kept up to w^4 (classify_exp bounds the rest over a whole block).
            const bool at_end = !(ua < 0.0);
            const float a = static_cast<float>(at_end ? -(L * rT) : L * rT);
            float ck = static_cast<float>(6.283185307179586 * (at_end ? -(f0s * exp(L)) : f0s)) * a * 0.5f;
            r.c2 = ck;
            ck *= a * (1.f / 3.f); r.c3 = ck;
            ck *= a * 0.25f; r.c4 = ck;
            r.kind = K_XEDGE;
            if (!at_end) {
                r.c5 = 1.f;
                r.c6 = static_cast<float>(-(ua + static_cast<double>(kHalf)));
                w = t.w_pre;
                ph = t.theta_pre + w * nc;
            } else {
                r.c5 = -1.f;
                r.c6 = static_cast<float>(-(Tn - ua - static_cast<double>(kHalf)));
                w = t.w_post;
                ph = t.theta_post + w * nc;
            }
        } else {
            // Whole block inside the move: phase and frequency at the block centre in fp64 (one expm1); the Taylor coefficients
            // of the phase are a geometric sequence, c_k = 2 pi (f/fs) a^(k-1) / k!.
            const double s = (ua + static_cast<double>(kHalf)) * rT;
            const double em = expm1(L * s);
            w = t.w_pre + frac_to_fix64(f0s * em);
            ph = t.theta_pre + t.w_pre * nc + frac_to_fix64(F * (em / L - s));
            const float a = static_cast<float>(L * rT);
            float ck = static_cast<float>(6.283185307179586 * f0s * (em + 1.0)) * a * 0.5f;
            r.c2 = ck;
            r.kind = K_QUAD;
            if (c >= CLS_DEG4) {
                ck *= a * (1.f / 3.f); r.c3 = ck;
                ck *= a * 0.25f; r.c4 = ck;
                r.kind = K_DEG4;
                if (c >= CLS_DEG6) {
                    ck *= a * 0.2f; r.c5 = ck;
                    ck *= a * (1.f / 6.f); r.c6 = ck;
                    r.kind = K_DEG6;
                }
            }
        }
    }
    r.c0 = round32(ph);
    r.c1 = round32(w);
    return r;
}

// Step a1.  Lane-private: tone record `rec` (index t) at the block whose first sample is blk_base (absolute);
// bb_d = (double)blk_base, nc = blk_base + kHalf.
__device__ __forceinline__ BlockRec block_prologue(const ToneRec *rec, int t, uint64_t nc, double bb_d)
{
    BlockRec r;
    r.c2 = r.c3 = r.c4 = r.c5 = r.c6 = 0.f;
    r.kind = K_STATIC;
    const uint4 v0 = ldg16(rec);  // A, cls, theta_pre
    r.A = __uint_as_float(v0.x);
    const int32_t cls = static_cast<int32_t>(v0.y);
    const int c = cls & 0xff;
    const uint64_t theta_pre = u64_of(v0.z, v0.w);
    const uint4 v1 = ldg16(reinterpret_cast<const char *>(rec) + 16);  // w_pre, theta_post
    // all seven loads are issued before the first use: one memory round trip per record instead of three
    const uint4 v2 = ldg16(reinterpret_cast<const char *>(rec) + 32);  // w_post, ns_int
    const uint4 v3 = ldg16(reinterpret_cast<const char *>(rec) + 48);  // ns_frac, Tn
    const uint4 v4 = ldg16(reinterpret_cast<const char *>(rec) + 64);  // inv_Tn, DT
    const uint4 v5 = ldg16(reinterpret_cast<const char *>(rec) + 80);  // q1, q[0], q[1]
    const uint4 v6 = ldg16(reinterpret_cast<const char *>(rec) + 96);  // q[2], q[3], q[4], A1
    const uint64_t w_pre = u64_of(v1.x, v1.y);
    if (cls & CLS_AMP_FLAG) {
        // amplitude ramp: a block it overlaps is evaluated per sample (K_EXACT), one after it takes A1
        const uint4 v7 = ldg16(reinterpret_cast<const char *>(rec) + 112);  // amp_ns, amp_Tn, amp_prof
        const double aa = bb_d - f64_of(v7.x, v7.y);
        if (aa >= static_cast<double>(__uint_as_float(v7.z))) {
            r.A = __uint_as_float(v6.w);
        } else if (aa + static_cast<double>(kBlock - 1) > 0.0) {
            r.kind = K_EXACT;
            r.c0 = static_cast<uint32_t>(t);
            r.c1 = 0;
            return r;
        }
    }
    if (c != CLS_STATIC && c != CLS_EXACT && ((cls >> 8) & 0xff) == AWG_PROFILE_EXP) {
        const ExpRec er = exp_block(rec, c, nc, bb_d);
        r.c0 = er.kind == K_EXACT ? static_cast<uint32_t>(t) : er.c0;
        r.c1 = er.c1;
        r.c2 = er.c2; r.c3 = er.c3; r.c4 = er.c4; r.c5 = er.c5; r.c6 = er.c6;
        r.kind = er.kind;
        return r;
    }
    uint64_t ph, w;
    if (c == CLS_STATIC) {
        w = w_pre;
        ph = theta_pre + w * nc;
    } else {
        const double Tn = f64_of(v3.z, v3.w);
        const double ua = (bb_d - f64_of(v2.z, v2.w)) - f64_of(v3.x, v3.y);  // u of the block's first sample
        const double ub = ua + static_cast<double>(kBlock - 1);
        const bool linear = ((cls >> 8) & 0xff) == AWG_PROFILE_LINEAR;
        if (ub <= 0.0) {
            w = w_pre;
            ph = theta_pre + w * nc;
        } else if (ua >= Tn) {
            w = u64_of(v2.x, v2.y);
            ph = u64_of(v1.z, v1.w) + w * nc;
        } else if (c == CLS_EXACT || (ua < 0.0 && ub > Tn)) {
            r.kind = K_EXACT;
            r.c0 = static_cast<uint32_t>(t);
            r.c1 = 0;
            return r;
        } else {
            const double rT = f64_of(v4.x, v4.y);
            const double DT = f64_of(v4.z, v4.w);
            const float q2 = __uint_as_float(v5.z), q3 = __uint_as_float(v5.w);
            const float q4 = __uint_as_float(v6.x), q5 = __uint_as_float(v6.y), q6 = __uint_as_float(v6.z);
            if (ua >= 0.0 && ub <= Tn) {
                // whole block inside the move (g(0) = 0 and DT g(1) = post - pre, so the closed ends are included):
                // Taylor-expand DT*g((u_c + k)/Tn) about the block centre.  Phase and frequency (g, g') in fp64,
                // the higher derivatives only feed fp32 coefficients and are evaluated in fp32.
                const double s = (ua + static_cast<double>(kHalf)) * rT;
                const float sf = static_cast<float>(s);
                double g0, g1;
                if (linear) {
                    g0 = 0.5 * s * s; g1 = s;
                    r.c2 = q2;  // g'' = 1
                } else {
                    const double s2 = s * s;
                    g0 = s2 * s2 * (2.5 + s * (s - 3.0));
                    g1 = s2 * s * (10.0 + s * (6.0 * s - 15.0));
                    r.c2 = q2 * (sf * sf * (30.f + sf * (30.f * sf - 60.f)));
                }
                w = w_pre + frac_to_fix64(f64_of(v5.x, v5.y) * g1);  // instantaneous frequency at the block centre
                ph = theta_pre + w_pre * nc + frac_to_fix64(DT * g0);
                r.kind = K_QUAD;
                if (c >= CLS_DEG4) {
                    r.c3 = q3 * (sf * (60.f + sf * (120.f * sf - 180.f)));
                    r.c4 = q4 * (60.f + sf * (360.f * sf - 360.f));
                    r.kind = K_DEG4;
                    if (c >= CLS_DEG6) {
                        r.c5 = q5 * (720.f * sf - 360.f);
                        r.c6 = q6 * 720.f;
                        r.kind = K_DEG6;
                    }
                }
            } else {
                // exactly one end of the move lies inside the block.  With w the (clamped) distance into the move
                // from that end, both ends have the same polynomial: DT (w/Tn)^2/2 (LINEAR) or
                // DT (5/2 (w/Tn)^4 - 3 (w/Tn)^5 + (w/Tn)^6) (MINJERK) on top of the carrier valid outside the move
                // [at the end: g(1+x) - (1/2 + x) = 5/2 x^4 + 3 x^5 + x^6, x = -w/Tn].  q[k-2] = 2 pi DT/Tn^k/k!.
                if (linear) {
                    r.c2 = q2;                 // 2 pi DT/(2 Tn^2)
                } else {
                    r.c3 = q4 * 60.f;          // 2 pi DT 5/2 / Tn^4
                    r.c4 = q5 * -360.f;        // -3 * 2 pi DT / Tn^5
                    r.c5 = q6 * 720.f;         // 2 pi DT / Tn^6
                }
                if (ua < 0.0) {   // start inside: u = 0 at k = kb
                    r.kind = K_SBEG;
                    r.c6 = static_cast<float>(-(ua + static_cast<double>(kHalf)));
                    w = w_pre;
                    ph = theta_pre + w * nc;
                } else {          // end inside: u = Tn at k = kb; stored negated (w = max(kb - k, 0) = max(-k - (-kb), 0))
                    r.kind = K_SEND;
                    r.c6 = static_cast<float>(-(Tn - ua - static_cast<double>(kHalf)));
                    w = u64_of(v2.x, v2.y);
                    ph = u64_of(v1.z, v1.w) + w * nc;
                }
            }
        }
    }
    r.c0 = round32(ph);
    r.c1 = round32(w);
    return r;
}

// ---- shared memory of one warp ------------------------------------------------------------------------------
// One tile-static tone of the current batch (angle-addition pass; a thread owns 64 consecutive samples of the tile, four
// groups of 16): carrier phase (u32 turns) at the half-integer pair centre of group 0 of lane 16 [c0], per thread
// (64 samples) [c1] and per group (16 samples) [d], the rotation that carries a sine/cosine pair two groups on, and the
// tone's pair tables.
struct __align__(16) StageRec {
    uint32_t c0, c1, d, pad_;
    float r0, r1, r2, r3;        // static tone: {cos, sin}(2 pi 32 w), the rotation by two groups; slow mover: 2 c2, 3 c3
    float4 C03, C47, S03, S47;
    float4 bank_pad_;            // 112-byte stride: the 16-byte stores of eight lanes (one record each) fall on distinct banks
};
static_assert(sizeof(StageRec) == 112, "StageRec must be 112 bytes");

// One re-centred (tone, block) record of the MUFU pass: q[0] = {c0 bits, c1 bits, A, c2}; q[1] = {c3, c4, c5, c6}.
// K_EXACT: c0 = tone index.
struct __align__(16) MovRec {
    float4 q[2];
};

struct __align__(16) WarpSmem {
    StageRec st[kBatch + 2];                // +2: the loops prefetch one tone (one or two records) ahead
    MovRec mrec[kBatch + 1];                // +1: the loops prefetch one record ahead
    float4 park[kBlocksPerTile][kSPT / 4][32];   // the warp's static partial sums of the tile: [block][4 samples][lane]
    uint32_t mov[kMaxBatches];              // per batch of 32 tones: which ones take the MUFU pass in this tile
    uint32_t next;                          // (rank-0 warp of a team) the team's next tile, drawn by the leader
    uint32_t n_mov;                         // how many of the warp's tones take the MUFU pass in this tile
    uint32_t last;                          // (warp 0) this CTA delivered the last quad of its tile: it sums and stores
    uint32_t pad_[1];
    uint16_t nm_leaf[kMaxQuads];            // per leaf of the warp: how many of its tones take the MUFU pass in this tile
    uint16_t list[kListCap];                // compacted tone indices of the MUFU pass (n_tones <= 65536)
};

// 16 samples of one block of one thread, as 8 packed pairs: a[j] = samples (2j, 2j+1).
struct Acc16 {
    float2 a[kPairs];
};

// The park area is indexed [block][4 samples][column] in the BLOCK layout of the MUFU pass and of the stores (thread
// `lane` of block r holds samples lane*16 .. +15 of the block).  The angle-addition passes work in the GROUP layout: a
// thread owns 64 consecutive samples of the tile, four groups of 16, so its group g is what thread
// lane' = (lane % 8) * 4 + g of block lane / 8 holds in the block layout.  park_col() swizzles the column so that both
// the group-layout writers (column stride 4 across lanes) and the block-layout readers are free of bank conflicts.
__device__ __forceinline__ int park_col(int lane_blk) { return lane_blk ^ (lane_blk >> 3); }
__device__ __forceinline__ int group_block(int lane) { return lane >> 3; }
__device__ __forceinline__ int group_col(int lane, int g) { return park_col(((lane & 7) << 2) | g); }

// group layout: the 16 samples of group g of this thread
__device__ __forceinline__ void park_store(WarpSmem &ws, int g, int lane, const Acc16 &acc)
{
    const int r = group_block(lane), col = group_col(lane, g);
#pragma unroll
    for (int v = 0; v < kSPT / 4; ++v)
        ws.park[r][v][col] = make_float4(acc.a[2 * v].x, acc.a[2 * v].y, acc.a[2 * v + 1].x, acc.a[2 * v + 1].y);
}

// block layout: the 16 samples of this thread in block r
__device__ __forceinline__ void park_load(const WarpSmem &ws, int r, int lane, Acc16 &acc)
{
    const int col = park_col(lane);
#pragma unroll
    for (int v = 0; v < kSPT / 4; ++v) {
        const float4 u = ws.park[r][v][col];
        acc.a[2 * v] = make_float2(u.x, u.y);
        acc.a[2 * v + 1] = make_float2(u.z, u.w);
    }
}

__device__ __forceinline__ void park_add(const WarpSmem &ws, int r, int lane, Acc16 &acc)
{
    const int col = park_col(lane);
#pragma unroll
    for (int v = 0; v < kSPT / 4; ++v) {
        const float4 u = ws.park[r][v][col];
        acc.a[2 * v].x += u.x; acc.a[2 * v].y += u.y;
        acc.a[2 * v + 1].x += u.z; acc.a[2 * v + 1].y += u.w;
    }
}

// Even/odd accumulators of the angle-addition pass for one block: sample (8 + j) = P_j + Q_j, sample (7 - j) = P_j - Q_j.
struct PQ {
    float2 P[kPairs / 2], Q[kPairs / 2];  // pairs (j, j+1), j = 0, 2, 4, 6
};

// Fixed-point merge of large tables (awg::tone_groups, FixGrid): a leaf's fp32 sums are rounded once to the leaf's grid
// -- fma(v, 2^sh, 1.5 * 2^23) leaves the integer in the low mantissa bits, |v 2^sh| < 2^22 by the host's choice of sh --
// and shifted on to the table's common grid; from there on everything is added in integers: exact, so the order in
// which leaves, warps and CTAs meet does not matter.
constexpr int kMagicBits = 0x4B400000;   // bits of 1.5 * 2^23

__device__ __forceinline__ float pow2f(int e) { return __int_as_float((127 + e) << 23); }

__device__ __forceinline__ int fix_of(float t, int mul) { return (__float_as_int(t) - kMagicBits) * mul; }

// The even/odd accumulators P_j, Q_j of one block of a leaf join the warp's leaves in its park area (int32 on the common
// grid).  The magic-number bias stays in: new = bits * mul + old is one IMAD per value, and the bias, kMagicBits * (sum
// of the leaves' mul), is taken out once when the team's park areas are added up (FixGrid::bias_q; integer arithmetic
// wraps, so this is exact).  The samples P_j +- Q_j are formed there too, in integers.
__device__ __forceinline__ void ipark_leaf(WarpSmem &ws, int g, int lane, const PQ &pq, float fscale, int mul, bool first)
{
    const int r = group_block(lane), col = group_col(lane, g);   // group layout -> the block layout of the park area
    const float2 sc = dup2(fscale), mg = dup2(kRoundMagic);
#pragma unroll
    for (int v = 0; v < kSPT / 4; ++v) {
        const float2 a = v < 2 ? pq.P[2 * v] : pq.Q[2 * v - 4], b = v < 2 ? pq.P[2 * v + 1] : pq.Q[2 * v - 3];
        const float2 t0 = __ffma2_rn(a, sc, mg), t1 = __ffma2_rn(b, sc, mg);
        int4 *slot = reinterpret_cast<int4 *>(&ws.park[r][v][col]);
        int4 u = make_int4(0, 0, 0, 0);
        if (!first) u = *slot;
        *slot = make_int4(__float_as_int(t0.x) * mul + u.x, __float_as_int(t0.y) * mul + u.y, __float_as_int(t1.x) * mul + u.z,
                          __float_as_int(t1.y) * mul + u.w);
    }
}

// i[0..7] = P_0..P_7, i[8..15] = Q_0..Q_7 (bias removed) -> the block's 16 samples: (8 + j) = P_j + Q_j, (7 - j) = P_j - Q_j
__device__ __forceinline__ void ipq_to_samples(const int (&i)[kSPT], int (&smp)[kSPT])
{
#pragma unroll
    for (int j = 0; j < kPairs; ++j) {
        smp[kPairs + j] = i[j] + i[kPairs + j];
        smp[kPairs - 1 - j] = i[j] - i[kPairs + j];
    }
}

__device__ __forceinline__ void ipark_add(const WarpSmem &ws, int r, int lane, int (&isum)[kSPT])
{
    const int col = park_col(lane);
#pragma unroll
    for (int v = 0; v < kSPT / 4; ++v) {
        const int4 u = *reinterpret_cast<const int4 *>(&ws.park[r][v][col]);
        isum[4 * v] += u.x; isum[4 * v + 1] += u.y; isum[4 * v + 2] += u.z; isum[4 * v + 3] += u.w;
    }
}

// Steps a2-a4, MUFU path, for ONE record of kind KIND.  Samples go in pairs through the packed fp32x2
// instructions of sm_100 (FMUL2 / FFMA2: one issue slot for two samples); the 16 sine chains are independent.
template <int KIND>
__device__ __forceinline__ void mufu_rec(const float4 a, const float4 b, int koff, const float2 (&kfs)[kPairs],
                                         const float2 (&kks)[kPairs], Acc16 &acc)
{
    const float2 K2 = dup2(kTurnToRad);
    const uint32_t c0 = __float_as_uint(a.x), c1 = __float_as_uint(a.y);
    const float A = a.z;
    const uint32_t base = c0 + c1 * static_cast<uint32_t>(koff);
#pragma unroll
    for (int j = 0; j < kPairs; ++j) {
        const uint32_t p0 = base + c1 * static_cast<uint32_t>(2 * j);
        const uint32_t p1 = base + c1 * static_cast<uint32_t>(2 * j + 1);
        const float2 f = make_float2(__int2float_rn(static_cast<int32_t>(p0)), __int2float_rn(static_cast<int32_t>(p1)));
        const float2 kf = kfs[j];
        float2 x;
        if (KIND == K_STATIC) {
            x = __fmul2_rn(f, K2);
        } else if (KIND == K_SBEG || KIND == K_SEND) {
            float2 w;
            w.x = fmaxf((KIND == K_SBEG ? kf.x : -kf.x) - b.w, 0.f);
            w.y = fmaxf((KIND == K_SBEG ? kf.y : -kf.y) - b.w, 0.f);
            const float2 w2 = __fmul2_rn(w, w);
            float2 poly = __ffma2_rn(dup2(b.z), w, dup2(b.y));
            poly = __ffma2_rn(poly, w, dup2(b.x));
            poly = __ffma2_rn(poly, w2, dup2(a.w));
            x = __ffma2_rn(f, K2, __fmul2_rn(poly, w2));
        } else if (KIND == K_XEDGE) {
            float2 w;
            w.x = fmaxf(fmaf(b.z, kf.x, -b.w), 0.f);
            w.y = fmaxf(fmaf(b.z, kf.y, -b.w), 0.f);
            const float2 w2 = __fmul2_rn(w, w);
            float2 poly = __ffma2_rn(dup2(b.y), w, dup2(b.x));
            poly = __ffma2_rn(poly, w, dup2(a.w));
            x = __ffma2_rn(f, K2, __fmul2_rn(poly, w2));
        } else {
            const float2 kk = kks[j];
            float2 poly;
            if (KIND == K_QUAD) {
                poly = dup2(a.w);
            } else if (KIND == K_DEG4) {
                poly = __ffma2_rn(dup2(b.y), kf, dup2(b.x));
                poly = __ffma2_rn(poly, kf, dup2(a.w));
            } else {
                poly = __ffma2_rn(dup2(b.w), kf, dup2(b.z));
                poly = __ffma2_rn(poly, kf, dup2(b.y));
                poly = __ffma2_rn(poly, kf, dup2(b.x));
                poly = __ffma2_rn(poly, kf, dup2(a.w));
            }
            x = __ffma2_rn(f, K2, __fmul2_rn(poly, kk));
        }
        acc.a[j] = __ffma2_rn(dup2(A), make_float2(mufu_sin(x.x), mufu_sin(x.y)), acc.a[j]);
    }
}

// fp64 path for a K_EXACT record (tones whose fp32 polynomial would be inaccurate, moves shorter than a block,
// instant retunes, blocks inside an amplitude ramp): exact phase and amplitude per sample, same sine.
__device__ __noinline__ Acc16 exact_rec(const ToneRec *tab, const float4 a, int64_t n_thread, Acc16 acc)
{
    const ToneCore &tr = tab[__float_as_uint(a.x)].core;
#pragma unroll 1
    for (int j = 0; j < kPairs; ++j) {
        const uint32_t p0 = round32(exact_phase(tr, n_thread + 2 * j));
        const uint32_t p1 = round32(exact_phase(tr, n_thread + 2 * j + 1));
        float2 v = acc.a[0];
        // rotate through the pairs so that the loop body indexes a[] statically
        v.x = fmaf(amp_at(tr, n_thread + 2 * j), mufu_sin(__int2float_rn(static_cast<int32_t>(p0)) * kTurnToRad), v.x);
        v.y = fmaf(amp_at(tr, n_thread + 2 * j + 1), mufu_sin(__int2float_rn(static_cast<int32_t>(p1)) * kTurnToRad), v.y);
#pragma unroll
        for (int m = 0; m < kPairs - 1; ++m) acc.a[m] = acc.a[m + 1];
        acc.a[kPairs - 1] = v;
    }
    return acc;
}

// Step a5 for 8 consecutive samples: v -> int16 code = clamp(rint_half_even(scale*v), -32768, 32767), packed into 16 bytes.
// The clamp is applied to v (bounds -32768/scale, 32767/scale: qlo, qhi); the fused multiply-add against 1.5*2^23 then
// rounds scale*v ONCE, to nearest-even, into the low mantissa bits: the two's-complement code is the low half-word.
// Runs on the ALU and FMA pipes (a float-to-int conversion would take the XU pipe the sines need).
__device__ __forceinline__ uint4 pack8(const LaunchParams &lp, const float2 (&s)[4])
{
    uint32_t w[4];
    const float2 sc = dup2(lp.scale), mg = dup2(kRoundMagic);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float2 v = make_float2(fminf(fmaxf(s[j].x, lp.qlo), lp.qhi), fminf(fmaxf(s[j].y, lp.qlo), lp.qhi));
        const float2 t = __ffma2_rn(v, sc, mg);
        w[j] = __byte_perm(__float_as_uint(t.x), __float_as_uint(t.y), 0x5410);
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}

// Steps a5-a6 for one block of one thread: 16 consecutive samples starting at absolute index n_thread, as two
// 8-sample halves (launch ranges are multiples of 8 samples, so each half is inside or outside as a whole).
// xs_tile: position of the tile's first sample in the looped static buffer (Eq. 9: X_static[i mod L_s] is added
// before quantisation); tile_off = n_thread - tile_base.
__device__ __forceinline__ void store_block(const LaunchParams &lp, int64_t n_thread, int64_t xs_tile, int tile_off, const Acc16 &acc)
{
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int64_t off = n_thread + 8 * h - lp.n_begin;
        if (off < 0 || off >= lp.n_count) continue;
        float2 a[4] = {acc.a[4 * h], acc.a[4 * h + 1], acc.a[4 * h + 2], acc.a[4 * h + 3]};
        if (lp.xs) {
            int64_t i = xs_tile + tile_off + 8 * h;     // < 2 L_s: one wrap at most (L_s >= kTile)
            if (i >= lp.xs_len) i -= lp.xs_len;
            const float4 x0 = __ldg(reinterpret_cast<const float4 *>(lp.xs + i)), x1 = __ldg(reinterpret_cast<const float4 *>(lp.xs + i) + 1);
            a[0].x += x0.x; a[0].y += x0.y; a[1].x += x0.z; a[1].y += x0.w;
            a[2].x += x1.x; a[2].y += x1.y; a[3].x += x1.z; a[3].y += x1.w;
        }
        if (lp.out_f32) {
            float4 *o = reinterpret_cast<float4 *>(static_cast<float *>(lp.out) + off);
            o[0] = make_float4(a[0].x, a[0].y, a[1].x, a[1].y);
            o[1] = make_float4(a[2].x, a[2].y, a[3].x, a[3].y);
        } else {
            const uint4 w = pack8(lp, a);
            if (lp.out_stride == 1) {
                *reinterpret_cast<uint4 *>(static_cast<int16_t *>(lp.out) + off) = w;
            } else {
                // multiplexed channels (the paper's WM): this channel's code of every sample index
                uint16_t *o = static_cast<uint16_t *>(lp.out) + off * lp.out_stride + lp.out_offset;
                const int st = lp.out_stride;
                o[0] = static_cast<uint16_t>(w.x); o[st] = static_cast<uint16_t>(w.x >> 16);
                o[2 * st] = static_cast<uint16_t>(w.y); o[3 * st] = static_cast<uint16_t>(w.y >> 16);
                o[4 * st] = static_cast<uint16_t>(w.z); o[5 * st] = static_cast<uint16_t>(w.z >> 16);
                o[6 * st] = static_cast<uint16_t>(w.w); o[7 * st] = static_cast<uint16_t>(w.w >> 16);
            }
        }
    }
}

__device__ __forceinline__ void pq_add(PQ &pq, float s, float c, const float4 &C03, const float4 &C47, const float4 &S03,
                                       const float4 &S47)
{
    const float2 s2 = dup2(s), c2 = dup2(c);
    pq.P[0] = __ffma2_rn(s2, make_float2(C03.x, C03.y), pq.P[0]);
    pq.P[1] = __ffma2_rn(s2, make_float2(C03.z, C03.w), pq.P[1]);
    pq.P[2] = __ffma2_rn(s2, make_float2(C47.x, C47.y), pq.P[2]);
    pq.P[3] = __ffma2_rn(s2, make_float2(C47.z, C47.w), pq.P[3]);
    pq.Q[0] = __ffma2_rn(c2, make_float2(S03.x, S03.y), pq.Q[0]);
    pq.Q[1] = __ffma2_rn(c2, make_float2(S03.z, S03.w), pq.Q[1]);
    pq.Q[2] = __ffma2_rn(c2, make_float2(S47.x, S47.y), pq.Q[2]);
    pq.Q[3] = __ffma2_rn(c2, make_float2(S47.z, S47.w), pq.Q[3]);
}

__device__ __forceinline__ Acc16 pq_to_samples(const PQ &pq)
{
    Acc16 d;
#pragma unroll
    for (int m = 0; m < kPairs / 2; ++m) {
        const float2 p = pq.P[m], q = pq.Q[m];              // j = 2m, 2m+1
        d.a[4 + m] = make_float2(p.x + q.x, p.y + q.y);      // samples 8 + 2m, 9 + 2m
        d.a[3 - m] = make_float2(p.y - q.y, p.x - q.x);      // samples 6 - 2m, 7 - 2m
    }
    return d;
}

// Loads the carrier part of a tone record (A, cls, theta_pre | w_pre, theta_post | w_post, ns_int | ns_frac, Tn).
__device__ __forceinline__ void fetch_tone(const ToneRec *tr, uint4 &v0, uint4 &v1, uint4 &v2, uint4 &v3)
{
    const char *p = reinterpret_cast<const char *>(tr);
    v0 = ldg16(p);
    v1 = ldg16(p + 16);
    v2 = ldg16(p + 32);
    v3 = ldg16(p + 48);
}

// Pulls a tone record (carrier part and the two angle-addition tables, bytes 0..63 and 128..287) towards L1: issued one
// batch ahead, so that the loads of the next batch's staging hit L1 and no register stays live across the multiply-add loop.
__device__ __forceinline__ void prefetch_tone(const ToneRec *tr)
{
    const char *p = reinterpret_cast<const char *>(tr);
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p + 128));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p + 208));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p + 272));
}

// Sines and cosines of one tile-static tone at the pair centres of the thread's four groups of 16 samples.
// rec header = {phase at the centre of group 0 of lane 16, phase per thread (64 samples), phase per group (16), - | cos,
// sin of the phase of two groups}; l16 = lane - 16.  Groups 0 and 1 come from MUFU (u32 turns -> radians -> sin.approx,
// cos.approx); groups 2 and 3 are those two pairs rotated by two groups, (s, c) -> (s cd + c sd, c cd - s sd), four packed
// fp32 instructions for both: a sine/cosine chain through IADD, I2FP, FMUL, FMUL.RZ and two MUFU costs the multiply-add
// stream more issue slots than the rotation does (profiles/: pipe microbenchmarks).  The rotation constants are rounded
// once from fp64.
__device__ __forceinline__ void sincos_tile(const StageRec *rec, int l16, float (&s)[kBlocksPerTile], float (&c)[kBlocksPerTile])
{
    static_assert(kBlocksPerTile == 4, "sincos_tile serves four groups as two pairs");
    const uint4 cc = *reinterpret_cast<const uint4 *>(rec);
    const float2 rot = *reinterpret_cast<const float2 *>(&rec->r0);
    const uint32_t p0 = cc.x + cc.y * static_cast<uint32_t>(l16);
    const uint32_t p1 = p0 + cc.z;
    const float2 x01 = __fmul2_rn(make_float2(__int2float_rn(static_cast<int32_t>(p0)), __int2float_rn(static_cast<int32_t>(p1))), dup2(kTurnToRad));
    s[0] = mufu_sin(x01.x); c[0] = mufu_cos(x01.x);
    s[1] = mufu_sin(x01.y); c[1] = mufu_cos(x01.y);
    const float2 s01 = make_float2(s[0], s[1]), c01 = make_float2(c[0], c[1]);
    const float2 s23 = __ffma2_rn(c01, dup2(rot.y), __fmul2_rn(s01, dup2(rot.x)));
    const float2 c23 = __ffma2_rn(s01, dup2(-rot.y), __fmul2_rn(c01, dup2(rot.x)));
    s[2] = s23.x; s[3] = s23.y;
    c[2] = c23.x; c[3] = c23.y;
}

template <int SPLIT>
__device__ __forceinline__ void team_sync(int team)
{
    if (SPLIT == 1) __syncwarp();
    else if (SPLIT == kWarps) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(SPLIT * 32) : "memory");
}

// MUFU pass of one warp over ONE BLOCK of a tile, for the tones the team's warps flagged in their `mov` bit masks
// (warp r2 owns tones r2*per ...).  The flagged tones of the whole team are compacted into ws.list (kListCap at a
// time); every listed tone is re-centred on the block (step a1, one lane per tone) and the records are then run
// KIND BY KIND (warp-uniform loops over ballot masks, no per-record switch) with one MUFU.SIN per tone-sample into
// the block's 16 samples per thread, which stay in registers.  Which records share a sub-batch depends only on the
// tile and the tone partition, never on the launch range, so the fp32 summation order is the same for every chunking.
#define AWG_RUN_KIND(K)                                                                  \
    {                                                                                    \
        const int e_ = kbase[K] + kcnt[K];                                               \
        if (kcnt[K] > 0) {                                                               \
            float4 a_ = ws.mrec[kbase[K]].q[0], b_ = ws.mrec[kbase[K]].q[1];             \
            _Pragma("unroll 1") for (int i_ = kbase[K] + 1; i_ <= e_; ++i_) {            \
                const float4 an_ = ws.mrec[i_].q[0], bn_ = ws.mrec[i_].q[1]; /* next record (slot kBatch: spare) */ \
                mufu_rec<K>(a_, b_, koff, kf, kk, acc);                                  \
                a_ = an_;                                                                \
                b_ = bn_;                                                                \
            }                                                                            \
        }                                                                                \
    }

template <int SPLIT>
__device__ __forceinline__ void mover_block(const LaunchParams &lp, WarpSmem &ws, const WarpSmem *team_ws, int r2_begin, int r2_end,
                                            int q, int per, int bpl, int64_t blk_base, int lane, Acc16 &acc)
{
    const int koff = lane * kSPT - kHalf;
    const unsigned lt = (1u << lane) - 1u;
    float2 kf[kPairs], kk[kPairs];  // in-block offsets k of the thread's samples, and k^2
#pragma unroll
    for (int j = 0; j < kPairs; ++j) {
        kf[j] = make_float2(static_cast<float>(koff + 2 * j), static_cast<float>(koff + 2 * j + 1));
        kk[j] = __fmul2_rn(kf[j], kf[j]);
    }
    // sources: leaf q (tones (q*SPLIT + r2)*per ..., batch masks mov[q*bpl ...]) of the team's warps r2_begin .. r2_end-1
    int r2 = r2_begin, b = 0;
    while (r2 < r2_end) {
        // gather: the moving tones of the team's warps, in (warp, tone) order, up to kListCap at a time
        int n = 0;
        while (r2 < r2_end && n + kBatch <= kListCap) {
            const int tb2 = min((q * SPLIT + r2) * per, lp.n_tones);   // first tone of warp r2's leaf q
            const int len = min(lp.n_tones, tb2 + per) - tb2;
            if (team_ws[r2].nm_leaf[q] == 0 || b * kBatch >= len) {
                ++r2;
                b = 0;
                continue;
            }
            const unsigned m = team_ws[r2].mov[q * bpl + b];
            if ((m >> lane) & 1u) ws.list[n + __popc(m & lt)] = static_cast<uint16_t>(tb2 + b * kBatch + lane);
            n += __popc(m);
            ++b;
        }
        if (n == 0) break;
        __syncwarp();
        for (int q0 = 0; q0 < n; q0 += kBatch) {
            BlockRec br;
            br.kind = K_NONE;
            if (q0 + lane < n) {
                const int t = ws.list[q0 + lane];
                br = block_prologue(lp.tab + t, t, static_cast<uint64_t>(blk_base + kHalf), static_cast<double>(blk_base));
            }
            const unsigned kv = __ballot_sync(0xffffffffu, br.kind >= 0);
            const unsigned k0 = __ballot_sync(0xffffffffu, (br.kind & 1) != 0);
            const unsigned k1 = __ballot_sync(0xffffffffu, (br.kind & 2) != 0);
            const unsigned k2 = __ballot_sync(0xffffffffu, (br.kind & 4) != 0);
            // records are stored sorted by kind, so every kind's records are contiguous: mrec[kbase[K] .. +kcnt[K])
            unsigned mk[K_COUNT];
            mk[K_STATIC] = kv & ~k0 & ~k1 & ~k2;
            mk[K_QUAD] = kv & k0 & ~k1 & ~k2;
            mk[K_DEG4] = kv & ~k0 & k1 & ~k2;
            mk[K_DEG6] = kv & k0 & k1 & ~k2;
            mk[K_SBEG] = kv & ~k0 & ~k1 & k2;
            mk[K_SEND] = kv & k0 & ~k1 & k2;
            mk[K_EXACT] = kv & ~k0 & k1 & k2;
            mk[K_XEDGE] = kv & k0 & k1 & k2;
            int kbase[K_COUNT], kcnt[K_COUNT];
            int slot = 0;
            {
                int run = 0;
#pragma unroll
                for (int k = 0; k < K_COUNT; ++k) {
                    kbase[k] = run;
                    kcnt[k] = __popc(mk[k]);
                    if (br.kind == k) slot = run + __popc(mk[k] & lt);
                    run += kcnt[k];
                }
            }
            __syncwarp();  // the previous sub-batch's readers are done
            if (br.kind >= 0) {
                ws.mrec[slot].q[0] = make_float4(__uint_as_float(br.c0), __uint_as_float(br.c1), br.A, br.c2);
                ws.mrec[slot].q[1] = make_float4(br.c3, br.c4, br.c5, br.c6);
            }
            __syncwarp();
            AWG_RUN_KIND(K_STATIC)
            AWG_RUN_KIND(K_QUAD)
            AWG_RUN_KIND(K_DEG4)
            AWG_RUN_KIND(K_DEG6)
            AWG_RUN_KIND(K_SBEG)
            AWG_RUN_KIND(K_SEND)
            AWG_RUN_KIND(K_XEDGE)
#pragma unroll 1
            for (int i_ = kbase[K_EXACT]; i_ < kbase[K_EXACT] + kcnt[K_EXACT]; ++i_)
                acc = exact_rec(lp.tab, ws.mrec[i_].q[0], blk_base + lane * kSPT, acc);
        }
        __syncwarp();  // ws.list is rebuilt for the next kListCap tones
    }
}
#undef AWG_RUN_KIND

// Serving order of the tiles: the launch's hot tiles (LaunchParams::hot, ascending) first, then the others in ascending order.
__device__ __forceinline__ int64_t hot_first(const LaunchParams &lp, int64_t seq)
{
    const int n_hot = lp.n_hot;
    if (n_hot == 0) return seq;
    if (seq < n_hot) return lp.hot[seq];
    int64_t t = seq - n_hot;
#pragma unroll 1
    for (int j = 0; j < n_hot && lp.hot[j] <= t; ++j) ++t;
    return t;
}

// Draws the team's next tile from the launch counter (leader: lane 0 of rank 0) and hands it to the whole team.
template <int SPLIT>
__device__ __forceinline__ int64_t next_unit(const LaunchParams &lp, WarpSmem &ws_leader, int team, int rank, int lane, int64_t n_teams)
{
    uint32_t v = 0;
    if (SPLIT == 1) {
        if (lane == 0) v = atomicAdd(lp.sched, 1u);
        v = __shfl_sync(0xffffffffu, v, 0);
    } else {
        if (rank == 0 && lane == 0) ws_leader.next = atomicAdd(lp.sched, 1u);
        team_sync<SPLIT>(team);
        v = ws_leader.next;
    }
    return n_teams + static_cast<int64_t>(v);
}

// Slow pass, staging (one lane per slow mover): the pair tables at the tile-centre frequency come from MUFU (the
// frequency changes from tile to tile, so they cannot be precomputed); the second record holds their derivatives with
// respect to the frequency, cos((j+1/2)(w + e)) ~ C_j - (j+1/2) e S_j,  sin((j+1/2)(w + e)) ~ S_j + (j+1/2) e C_j;
// the first record's header also carries the coefficients 2 c2 and 3 c3 of the local frequency offset
// e(k) = 2 c2 k + 3 c3 k^2 and the phase step of a group.
// parked: q[0] = {c0, phase per thread, c2, c3}, q[1] = {A, phase per group (bits), phase per sample (bits), -}
__device__ __forceinline__ void stage_slow(StageRec *dst, const MovRec &parked)
{
    const float4 a = parked.q[0];
    const uint32_t c1 = __float_as_uint(parked.q[1].z);
    const float A = parked.q[1].x;
    float C[kPairs], S[kPairs];
#pragma unroll
    for (int j = 0; j < kPairs; ++j) {
        const uint32_t ang = c1 * static_cast<uint32_t>(j) + (c1 >> 1);   // (j + 1/2) c1, u32 turns
        const float x = __int2float_rn(static_cast<int32_t>(ang)) * kTurnToRad;
        C[j] = A * mufu_cos(x);
        S[j] = A * mufu_sin(x);
    }
    *reinterpret_cast<float4 *>(&dst[0]) = a;
    *reinterpret_cast<float4 *>(&dst[0].r0) = make_float4(2.f * a.z, 3.f * a.w, parked.q[1].y, 0.f);
    dst[0].C03 = make_float4(C[0], C[1], C[2], C[3]);
    dst[0].C47 = make_float4(C[4], C[5], C[6], C[7]);
    dst[0].S03 = make_float4(S[0], S[1], S[2], S[3]);
    dst[0].S47 = make_float4(S[4], S[5], S[6], S[7]);
    // derivative record: dC_j/dw = -(j+1/2) S_j in the C slots, dS_j/dw = (j+1/2) C_j in the S slots
    dst[1].C03 = make_float4(-0.5f * S[0], -1.5f * S[1], -2.5f * S[2], -3.5f * S[3]);
    dst[1].C47 = make_float4(-4.5f * S[4], -5.5f * S[5], -6.5f * S[6], -7.5f * S[7]);
    dst[1].S03 = make_float4(0.5f * C[0], 1.5f * C[1], 2.5f * C[2], 3.5f * C[3]);
    dst[1].S47 = make_float4(4.5f * C[4], 5.5f * C[5], 6.5f * C[6], 7.5f * C[7]);
}

// Slow pass, per-thread constants: offsets (from the tile centre) of the pair centres of the thread's four groups,
// k_g = 64 (lane - 16) + 16 g + 7.5, packed over group pairs, their squares, and the offset of the thread's own centre.
struct SlowK {
    int l16;
    float kt;
    float2 kf01, kf23, kk01, kk23;
};

// Slow pass, one tone at one thread: sines and cosines of the cubic phase polynomial at the pair centres of the four
// groups (packed over group pairs: every fp32 instruction here serves two groups) and the tone's frequency offset from
// the tile-centre frequency at the thread's own centre, e = 2 c2 k + 3 c3 k^2.
struct SlowSC {
    float2 s01, s23, c01, c23;
    float e;         // at the thread's centre (one correction per thread) or at the centre of groups 0, 1
    float e_hi;      // two corrections per thread (SLOW2): at the centre of groups 2, 3
};

template <bool SLOW2>
__device__ __forceinline__ void slow_sincos(const StageRec *rec, const SlowK &K, SlowSC &o)
{
    const uint4 cc = *reinterpret_cast<const uint4 *>(rec);                 // c0, phase per thread, c2, c3
    const float4 g = *reinterpret_cast<const float4 *>(&rec->r0);           // 2 c2, 3 c3, phase per group (bits), -
    const float c2 = __uint_as_float(cc.z), c3 = __uint_as_float(cc.w);
    const uint32_t p0 = cc.x + cc.y * static_cast<uint32_t>(K.l16);
    const uint32_t db = __float_as_uint(g.z);
    const uint32_t p1 = p0 + db, p2 = p1 + db, p3 = p2 + db;
    static_assert(kBlocksPerTile == 4, "slow_sincos assumes four groups per thread");
    const float2 K2 = dup2(kTurnToRad);
    const float2 f01 = make_float2(__int2float_rn(static_cast<int32_t>(p0)), __int2float_rn(static_cast<int32_t>(p1)));
    const float2 f23 = make_float2(__int2float_rn(static_cast<int32_t>(p2)), __int2float_rn(static_cast<int32_t>(p3)));
    const float2 x01 = __ffma2_rn(f01, K2, __fmul2_rn(K.kk01, __ffma2_rn(K.kf01, dup2(c3), dup2(c2))));
    const float2 x23 = __ffma2_rn(f23, K2, __fmul2_rn(K.kk23, __ffma2_rn(K.kf23, dup2(c3), dup2(c2))));
    o.s01 = make_float2(mufu_sin(x01.x), mufu_sin(x01.y));
    o.c01 = make_float2(mufu_cos(x01.x), mufu_cos(x01.y));
    o.s23 = make_float2(mufu_sin(x23.x), mufu_sin(x23.y));
    o.c23 = make_float2(mufu_cos(x23.x), mufu_cos(x23.y));
    if (SLOW2) {
        const float klo = K.kt - static_cast<float>(kSPT), khi = K.kt + static_cast<float>(kSPT);
        o.e = klo * fmaf(klo, g.y, g.x);
        o.e_hi = khi * fmaf(khi, g.y, g.x);
    } else {
        o.e = K.kt * fmaf(K.kt, g.y, g.x);
    }
}

// Slow pass, the multiply-adds of one tone: the pair tables are moved to the thread's local frequency once,
// C'_j = C_j + e dC_j/dw, S'_j = S_j + e dS_j/dw (16 multiply-adds), and serve the thread's four groups (64): 1.25
// multiply-adds per tone-sample.
__device__ __forceinline__ void slow_tables(const StageRec *rec, float e, float4 &C03, float4 &C47, float4 &S03, float4 &S47)
{
    const float2 e2 = dup2(e);
    C03 = rec[0].C03; C47 = rec[0].C47; S03 = rec[0].S03; S47 = rec[0].S47;
    const float4 d0 = rec[1].C03, d1 = rec[1].C47, d2 = rec[1].S03, d3 = rec[1].S47;
    float2 t;
    t = __ffma2_rn(e2, make_float2(d0.x, d0.y), make_float2(C03.x, C03.y)); C03.x = t.x; C03.y = t.y;
    t = __ffma2_rn(e2, make_float2(d0.z, d0.w), make_float2(C03.z, C03.w)); C03.z = t.x; C03.w = t.y;
    t = __ffma2_rn(e2, make_float2(d1.x, d1.y), make_float2(C47.x, C47.y)); C47.x = t.x; C47.y = t.y;
    t = __ffma2_rn(e2, make_float2(d1.z, d1.w), make_float2(C47.z, C47.w)); C47.z = t.x; C47.w = t.y;
    t = __ffma2_rn(e2, make_float2(d2.x, d2.y), make_float2(S03.x, S03.y)); S03.x = t.x; S03.y = t.y;
    t = __ffma2_rn(e2, make_float2(d2.z, d2.w), make_float2(S03.z, S03.w)); S03.z = t.x; S03.w = t.y;
    t = __ffma2_rn(e2, make_float2(d3.x, d3.y), make_float2(S47.x, S47.y)); S47.x = t.x; S47.y = t.y;
    t = __ffma2_rn(e2, make_float2(d3.z, d3.w), make_float2(S47.z, S47.w)); S47.z = t.x; S47.w = t.y;
}

template <bool SLOW2>
__device__ __forceinline__ void slow_fma(const StageRec *rec, const SlowSC &v, PQ (&pq)[kBlocksPerTile])
{
    float4 C03, C47, S03, S47;
    slow_tables(rec, v.e, C03, C47, S03, S47);
    pq_add(pq[0], v.s01.x, v.c01.x, C03, C47, S03, S47);
    pq_add(pq[1], v.s01.y, v.c01.y, C03, C47, S03, S47);
    if (SLOW2) slow_tables(rec, v.e_hi, C03, C47, S03, S47);   // plans with faster slow movers: groups 2, 3 get their own local frequency (1.5 per tone-sample)
    pq_add(pq[2], v.s23.x, v.c23.x, C03, C47, S03, S47);
    pq_add(pq[3], v.s23.y, v.c23.y, C03, C47, S03, S47);
}

// A work unit is one 2048-sample tile (LEAVES launches with few tiles: one quad of tone leaves of a tile).  SPLIT warps (a
// team) share a tile, each taking 1/SPLIT of the tones; their partial sums meet in shared memory (the park areas).
// The grid is persistent (three CTAs per SM); teams start on the unit of their own index, team index = team_in_cta *
// gridDim.x + blockIdx.x, and then draw units from the launch's counter.
// ROT: tones that are static over the whole tile take the angle-addition pass (FMA engine), everything else (and
// every tone when !ROT) takes the MUFU pass.  Every sample goes through the same arithmetic for every launch
// geometry because all phases are anchored to absolute tile positions.
template <int SPLIT, bool ROT, bool LEAVES, bool SLOW2>
__global__ void __launch_bounds__(kWarps * 32, kCtasPerSm) awg_synth_kernel(const LaunchParams lp)
{
    constexpr int kTeams = kWarps / SPLIT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WarpSmem *ws_all = reinterpret_cast<WarpSmem *>(smem_raw);

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int team = warp / SPLIT;
    const int rank = warp % SPLIT;
    const unsigned lt = (1u << lane) - 1u;
    WarpSmem &ws = ws_all[warp];

    // tiles are anchored to absolute sample indices (chunk-size invariance, SURVEY.md 8(b) "Determinism")
    const int64_t first_tile = lp.n_begin / kTile;  // n_begin >= 0
    const int64_t n_end = lp.n_begin + lp.n_count;
    const int64_t n_tiles = (n_end - 1) / kTile - first_tile + 1;
    const int64_t n_teams = static_cast<int64_t>(gridDim.x) * kTeams;

    // Tone groups (awg::tone_groups): the tone table is cut into leaves of `per` tones; warp `rank` of a team takes the
    // leaves q*SPLIT + rank, q = 0 .. Q-1.  A leaf is summed FROM ZERO over its tones in tone order; a warp adds its
    // leaves in order (W_rank = ((l_0 + l_1) + l_2) ...), the team adds W_0 .. W_3 in rank order, and the moving tones of
    // every leaf are summed from zero per leaf and block and added leaf by leaf (S + M).  This fixed tree is what lets a
    // launch with few tiles hand the leaves of a tile to different CTAs (lp.cross) and still produce the same bits:
    // there the leaves meet in scratch memory and the CTA that delivers the last one adds them up in the same order.
    // Small tables (Q == 1) are one leaf per warp with the moving tones chained onto the static sum.
    constexpr bool kQuads = LEAVES;
    static_assert(!LEAVES || SPLIT == kWarps, "leaves are the large-table path: one CTA per team");
    const int per = lp.per;
    const int Q = kQuads ? lp.n_quads : 1;
    const int bpl = (per + kBatch - 1) / kBatch;   // batches per leaf
    const bool cross = kQuads && lp.cross != 0;
    const int64_t n_units = cross ? n_tiles * Q : n_tiles;
    const int l16 = lane - 16;   // angle-addition passes: the thread owns samples lane*64 .. +63 of the tile; phases are referenced to lane 16
    // Tile scheduler: every team starts on the tile of its own index and then draws tiles from the launch's
    // counter lp.sched[0] (tiles that hold moving tones cost several times the others, so a fixed stride leaves
    // SMs idle at the end).  Which team computes a tile has no effect on its samples.
    int64_t unit = static_cast<int64_t>(team) * gridDim.x + blockIdx.x;
    // The tone records of the next batch are pulled into L1 before the multiply-add loop of the current batch runs.
    // A warp whose tones fit one batch keeps their tables in shared memory for as long as the same tones are static on
    // the same carriers (sticky_sta / sticky_post).
    const bool single = !kQuads && per <= kBatch;
    unsigned sticky_sta = 0u, sticky_post = 0xffffffffu;   // no tile has post bits outside its static bits
    while (unit < n_units) {
      const int64_t tile_seq = cross ? unit / Q : unit;
      const int q_begin = cross ? static_cast<int>(unit - tile_seq * Q) : 0;
      const int64_t tile = hot_first(lp, tile_seq);
      const int q_end = cross ? q_begin + 1 : Q;
      const int64_t tile_base = (first_tile + tile) * kTile;
      const int64_t n_thread = tile_base + lane * kSPT;
      const int64_t xs_tile = lp.xs ? tile_base % lp.xs_len : 0;
      int n_mov_tile = 0;
#pragma unroll 1
      for (int q = q_begin; q < q_end; ++q) {
        const int t_begin = min((q * SPLIT + rank) * per, lp.n_tones);
        const int t_end = min(lp.n_tones, t_begin + per);
        uint32_t *const mov_q = ws.mov + q * bpl;
        Acc16 acc[kBlocksPerTile];
        int n_mov = 0;

        if (ROT) {
            // ---- angle-addition pass: tones that are static over the whole tile; the others are listed in ws.mov
            PQ pq[kBlocksPerTile];
#pragma unroll
            for (int r = 0; r < kBlocksPerTile; ++r)
#pragma unroll
                for (int m = 0; m < kPairs / 2; ++m) pq[r].P[m] = pq[r].Q[m] = make_float2(0.f, 0.f);
            const double tb_d = static_cast<double>(tile_base);
            // phase reference: the pair centre of group 0 of lane 16 (sample 16*64 + 8 of the tile, minus the half sample of the
            // pair centring); lanes are 64 samples apart, groups 16
            const uint64_t a0 = static_cast<uint64_t>(tile_base + kTile / 2 + kSPT / 2);
            for (int tb = t_begin, b = 0; tb < t_end; tb += kBatch, ++b) {
                const int t = tb + lane;
                bool is_static = false, is_mover = false, is_post = false, is_slow = false;
                uint32_t c0 = 0, c1 = 0, d = 0;
                const float4 *tabp = nullptr;
                if (t < t_end) {
                    const ToneRec *tr = lp.tab + t;
                    uint4 v0, v1, v2, v3;
                    fetch_tone(tr, v0, v1, v2, v3);
                    uint64_t th = u64_of(v0.z, v0.w), w = u64_of(v1.x, v1.y);
                    tabp = reinterpret_cast<const float4 *>(&tr->rot_pre);
                    is_static = true;
                    if ((static_cast<int32_t>(v0.y) & 0xff) != CLS_STATIC) {
                        const double ua = (tb_d - f64_of(v2.z, v2.w)) - f64_of(v3.x, v3.y);  // u of the tile's first sample
                        const double ub = ua + static_cast<double>(kTile - 1);
                        if (ub <= 0.0) {
                            // whole tile before the move: pre-move carrier
                        } else if (ua >= f64_of(v3.z, v3.w)) {
                            th = u64_of(v1.z, v1.w);
                            w = u64_of(v2.x, v2.y);
                            tabp = reinterpret_cast<const float4 *>(&tr->rot_post);
                            is_post = true;
                        } else if ((static_cast<int32_t>(v0.y) & CLS_SLOW_FLAG) && ua >= 0.0 && ub <= f64_of(v3.z, v3.w)) {
                            // Slow mover, tile wholly inside the move: cubic Taylor expansion of the phase about the tile
                            // centre (phase and frequency in u64 / fp64, curvature terms in fp32 radians); the record is
                            // parked in ws.mrec (free during the static pass) until the slow pass of this batch.
                            is_static = false;
                            is_slow = true;
                            const uint4 v4 = ldg16(reinterpret_cast<const char *>(tr) + 64);  // inv_Tn, DT
                            const uint4 v5 = ldg16(reinterpret_cast<const char *>(tr) + 80);  // q1, q[0], q[1]
                            const double sc = (ua + static_cast<double>(kTile / 2)) * f64_of(v4.x, v4.y);
                            const float sf = static_cast<float>(sc);
                            double g0, g1;
                            float g2, g3;
                            if (((static_cast<int32_t>(v0.y) >> 8) & 0xff) == AWG_PROFILE_LINEAR) {
                                g0 = 0.5 * sc * sc; g1 = sc; g2 = 1.f; g3 = 0.f;
                            } else {
                                const double s2 = sc * sc;
                                g0 = s2 * s2 * (2.5 + sc * (sc - 3.0));
                                g1 = s2 * sc * (10.0 + sc * (6.0 * sc - 15.0));
                                g2 = sf * sf * (30.f + sf * (30.f * sf - 60.f));
                                g3 = sf * (60.f + sf * (120.f * sf - 180.f));
                            }
                            const uint64_t nc = static_cast<uint64_t>(tile_base + kTile / 2);
                            const uint64_t wc = w + frac_to_fix64(f64_of(v5.x, v5.y) * g1);
                            const uint64_t pc = th + w * nc + frac_to_fix64(f64_of(v4.z, v4.w) * g0);
                            // linear part of the phase at the pair centre of group 0 of lane 16 (k = 7.5), per thread, per group, per sample
                            ws.mrec[lane].q[0] = make_float4(__uint_as_float(round32(pc + wc * static_cast<uint64_t>(kSPT / 2) - (wc >> 1))),
                                                             __uint_as_float(round32(wc * static_cast<uint64_t>(kBlocksPerTile * kSPT))),
                                                             __uint_as_float(v5.z) * g2, __uint_as_float(v5.w) * g3);
                            ws.mrec[lane].q[1] = make_float4(__uint_as_float(v0.x), __uint_as_float(round32(wc * static_cast<uint64_t>(kSPT))),
                                                             __uint_as_float(round32(wc)), 0.f);
                        } else {
                            is_static = false;
                            is_mover = true;
                            // the block owners re-centre this tone after the barrier: pull its record towards L1 now
                            asm volatile("prefetch.global.L1 [%0];" ::"l"(reinterpret_cast<const char *>(tr)));
                            asm volatile("prefetch.global.L1 [%0];" ::"l"(reinterpret_cast<const char *>(tr) + 96));
                        }
                    }
                    if (static_cast<int32_t>(v0.y) & CLS_AMP_FLAG) {
                        // amplitude ramp (Eq. 9's a_j[i]): the pre-move table carries A, the post-move table A1; a tile
                        // that is not wholly before (or after) both the move and the ramp takes the MUFU pass
                        const uint4 v7 = ldg16(reinterpret_cast<const char *>(tr) + 112);  // amp_ns, amp_Tn, amp_prof
                        const double aa = tb_d - f64_of(v7.x, v7.y);
                        const bool before = aa + static_cast<double>(kTile - 1) <= 0.0;
                        const bool after = aa >= static_cast<double>(__uint_as_float(v7.z));
                        if (is_static) {
                            if ((static_cast<int32_t>(v0.y) & 0xff) == CLS_STATIC && after) {
                                tabp = reinterpret_cast<const float4 *>(&tr->rot_post);
                                is_post = true;
                            } else if (is_post ? !after : !before) {
                                is_static = false;
                                is_mover = true;
                            }
                        } else if (is_slow) {
                            if (!before && !after) {
                                is_slow = false;
                                is_mover = true;
                            } else if (after) {
                                ws.mrec[lane].q[1].x = __ldg(&tr->core.A1);
                            }
                        }
                    }
                    c0 = round32(th + w * a0 - (w >> 1));
                    c1 = round32(w * static_cast<uint64_t>(kBlocksPerTile * kSPT));
                    d = round32(w * static_cast<uint64_t>(kSPT));
                }
                if (tb + kBatch < t_end) {
                    const int tn = tb + kBatch + lane;
                    if (tn < t_end) prefetch_tone(lp.tab + tn);
                } else if (q + 1 < q_end) {
                    // last batch of the leaf: the first batch of the warp's next leaf
                    const int tn0 = min(((q + 1) * SPLIT + rank) * per, lp.n_tones);
                    if (tn0 + lane < min(lp.n_tones, tn0 + per)) prefetch_tone(lp.tab + tn0 + lane);
                } else if (!single) {
                    // last batch of the tile: the first batch of the next one (the same tones unless the quads are spread over CTAs)
                    const int tn0 = min(rank * per, lp.n_tones);
                    if (!cross && tn0 + lane < min(lp.n_tones, tn0 + per)) prefetch_tone(lp.tab + tn0 + lane);
                }
                const unsigned m_mov = __ballot_sync(0xffffffffu, is_mover);
                const unsigned m_sta = __ballot_sync(0xffffffffu, is_static);
                const unsigned m_slow = __ballot_sync(0xffffffffu, is_slow);
                if (lane == 0) mov_q[b] = m_mov;
                n_mov += __popc(m_mov);
                const int n_sta = __popc(m_sta);
                __syncwarp();  // the previous batch's readers are done
                const unsigned m_post = __ballot_sync(0xffffffffu, is_post);
                const bool tables_staged = single && m_sta == sticky_sta && m_post == sticky_post;
                sticky_sta = m_sta;
                sticky_post = m_post;
                if (is_static) {
                    StageRec &sr = ws.st[__popc(m_sta & lt)];
                    *reinterpret_cast<uint4 *>(&sr) = make_uint4(c0, c1, d, 0u);
                    if (!tables_staged) {
                        const float4 C03 = __ldg(tabp), C47 = __ldg(tabp + 1), S03 = __ldg(tabp + 2), S47 = __ldg(tabp + 3);
                        const float4 R = __ldg(tabp + 4);   // {cos, sin}(two blocks of phase), -, -
                        sr.C03 = C03; sr.C47 = C47; sr.S03 = S03; sr.S47 = S47;
                        *reinterpret_cast<float4 *>(&sr.r0) = R;
                    }
                }
                __syncwarp();
                // Software pipeline, unrolled by two so that the sines/cosines ping-pong between two register sets:
                // the phase -> I2FP -> FMUL2 -> MUFU chain of tone i+1 (XU and ALU pipes) is issued under the
                // 32 FFMA2 of tone i.  Scalar fp32 instructions cost the FMA pipe as much as an FFMA2 (measured,
                // profiles/), hence the packed range multiply and no register moves.
                float sa[kBlocksPerTile], ca[kBlocksPerTile], sb[kBlocksPerTile], cb[kBlocksPerTile];
                sincos_tile(&ws.st[0], l16, sa, ca);
                // a running pointer keeps the loop free of index arithmetic (IMAD shares the FMA pipe)
                const StageRec *sp = ws.st;
                const StageRec *const sp_end = ws.st + n_sta;
#pragma unroll 1
                for (; sp + 1 < sp_end; sp += 2) {
                    {
                        const float4 C03 = sp[0].C03, C47 = sp[0].C47, S03 = sp[0].S03, S47 = sp[0].S47;
                        sincos_tile(sp + 1, l16, sb, cb);
#pragma unroll
                        for (int r = 0; r < kBlocksPerTile; ++r) pq_add(pq[r], sa[r], ca[r], C03, C47, S03, S47);
                    }
                    {
                        const float4 C03 = sp[1].C03, C47 = sp[1].C47, S03 = sp[1].S03, S47 = sp[1].S47;
                        // slot i + 2 <= kBatch exists; past the last tone it is stale and its result unused
                        sincos_tile(sp + 2, l16, sa, ca);
#pragma unroll
                        for (int r = 0; r < kBlocksPerTile; ++r) pq_add(pq[r], sb[r], cb[r], C03, C47, S03, S47);
                    }
                }
                if (sp < sp_end) {
                    const float4 C03 = sp[0].C03, C47 = sp[0].C47, S03 = sp[0].S03, S47 = sp[0].S47;
#pragma unroll
                    for (int r = 0; r < kBlocksPerTile; ++r) pq_add(pq[r], sa[r], ca[r], C03, C47, S03, S47);
                }
                // ---- slow pass: the batch's slow movers, 16 lanes at a time (two staged records per tone: the tone
                // at the tile-centre frequency, and the first-order correction of its pair tables)
                if (m_slow != 0u) {
                    SlowK slowk;
                    {
                        slowk.l16 = l16;
                        const float k0 = static_cast<float>(l16 * (kBlocksPerTile * kSPT)) + (0.5f * kSPT - 0.5f);   // group 0: 64 (lane - 16) + 7.5
                        slowk.kf01 = make_float2(k0, k0 + static_cast<float>(kSPT));
                        slowk.kf23 = make_float2(k0 + static_cast<float>(2 * kSPT), k0 + static_cast<float>(3 * kSPT));
                        slowk.kk01 = __fmul2_rn(slowk.kf01, slowk.kf01);
                        slowk.kk23 = __fmul2_rn(slowk.kf23, slowk.kf23);
                        slowk.kt = static_cast<float>(l16 * (kBlocksPerTile * kSPT)) + (0.5f * (kBlocksPerTile * kSPT) - 0.5f);   // the thread's centre: + 31.5
                    }
                    sticky_sta = 0u;           // ws.st is overwritten: a single-batch warp restages its tables next tile
                    sticky_post = 0xffffffffu;
#pragma unroll 1
                    for (int half = 0; half < 2; ++half) {
                        const unsigned mh = m_slow & (0xffffu << (16 * half));
                        if (mh == 0u) continue;
                        __syncwarp();  // the readers of ws.st are done
                        if (is_slow && (lane >> 4) == half) stage_slow(ws.st + 2 * __popc(mh & lt), ws.mrec[lane]);
                        __syncwarp();
                        // software pipeline over the half's tones, unrolled by two (ping-pong register sets): the phase
                        // polynomial, sines and cosines of tone i+1 are issued under the 64 FFMA2 of tone i
                        const StageRec *sp = ws.st;
                        const StageRec *const sp_end = ws.st + 2 * __popc(mh);
                        SlowSC va, vb;
                        slow_sincos<SLOW2>(sp, slowk, va);
#pragma unroll 1
                        for (; sp + 2 < sp_end; sp += 4) {
                            slow_sincos<SLOW2>(sp + 2, slowk, vb);
                            slow_fma<SLOW2>(sp, va, pq);
                            slow_sincos<SLOW2>(sp + 4, slowk, va);   // slots up to 2*16 + 1 exist; past the last tone: stale, unused
                            slow_fma<SLOW2>(sp + 2, vb, pq);
                        }
                        if (sp < sp_end) slow_fma<SLOW2>(sp, va, pq);
                    }
                }
            }
            if (kQuads) {
                // the leaf's sums, rounded to the leaf's fixed-point grid, join the warp's leaves in its park area (int32)
                const int sh = lp.fix.leaf_sh[q * 4 + rank];
#pragma unroll
                for (int r = 0; r < kBlocksPerTile; ++r) ipark_leaf(ws, r, lane, pq[r], pow2f(sh), 1 << (lp.fix.fix_sh - sh), q == q_begin);
            } else {
#pragma unroll
                for (int r = 0; r < kBlocksPerTile; ++r) acc[r] = pq_to_samples(pq[r]);
            }
        } else {
            for (int tb = t_begin, b = 0; tb < t_end; tb += kBatch, ++b) {
                const int left = t_end - tb;
                if (lane == 0) mov_q[b] = left >= 32 ? 0xffffffffu : ((1u << left) - 1u);
            }
            n_mov = max(t_end - t_begin, 0);
        }

        if (lane == 0) ws.nm_leaf[q] = static_cast<uint16_t>(min(n_mov, 65535));
        n_mov_tile += n_mov;
        if (!kQuads) {
            if (SPLIT == 1 && ROT && n_mov == 0) {
#pragma unroll
                for (int g = 0; g < kBlocksPerTile; ++g) park_store(ws, g, lane, acc[g]);
                __syncwarp();
                // (through the park area: group layout -> block layout, whose 16-byte stores are contiguous across the warp)
#pragma unroll
                for (int r = 0; r < kBlocksPerTile; ++r) {
                    Acc16 blk;
                    park_load(ws, r, lane, blk);
                    store_block(lp, n_thread + r * kBlock, xs_tile, lane * kSPT + r * kBlock, blk);
                }
                __syncwarp();
            } else if (ROT) {
#pragma unroll
                for (int r = 0; r < kBlocksPerTile; ++r) park_store(ws, r, lane, acc[r]);
            }
        }
      }

      if (!(SPLIT == 1 && ROT && n_mov_tile == 0)) {
        // ---- the static partial sums and the lists of moving tones are in shared memory; after the team barrier
        // warp `rank` owns the blocks rank, rank + SPLIT, ...: it adds the team's partial sums, runs the MUFU pass of
        // that block for the moving tones of EVERY warp of the team (so the moving tones load the team's warps evenly
        // wherever they sit in the tone table), quantises and stores.
        if (lane == 0) ws.n_mov = static_cast<uint32_t>(n_mov_tile);
        team_sync<SPLIT>(team);
        WarpSmem *team_ws = ws_all + (warp - rank);
#pragma unroll 1
        for (int r = rank; r < kBlocksPerTile; r += SPLIT) {
            const int64_t blk_base = tile_base + static_cast<int64_t>(r) * kBlock;
            if (blk_base >= n_end || blk_base + kBlock <= lp.n_begin) continue;
            uint32_t any = 0;
#pragma unroll
            for (int r2 = 0; r2 < SPLIT; ++r2) any |= team_ws[r2].n_mov;
            if (!kQuads) {
                // small tables: fp32 all the way, partial sums in rank order, the moving tones chained on top
                Acc16 sum;
#pragma unroll
                for (int j = 0; j < kPairs; ++j) sum.a[j] = make_float2(0.f, 0.f);
                if (ROT) {
#pragma unroll
                    for (int r2 = 0; r2 < SPLIT; ++r2) park_add(team_ws[r2], r, lane, sum);
                }
                if (any) mover_block<SPLIT>(lp, ws, team_ws, 0, SPLIT, 0, per, bpl, blk_base, lane, sum);
                store_block(lp, n_thread + r * kBlock, xs_tile, lane * kSPT + r * kBlock, sum);
            } else {
                // large tables: leaves and per-quad moving-tone sums meet in fixed point (exact, any order)
                int isum[kSPT];
#pragma unroll
                for (int j = 0; j < kSPT; ++j) isum[j] = 0;
                if (ROT) {
                    int ipq[kSPT];
#pragma unroll
                    for (int j = 0; j < kSPT; ++j) ipq[j] = 0;
#pragma unroll
                    for (int r2 = 0; r2 < SPLIT; ++r2) ipark_add(team_ws[r2], r, lane, ipq);
                    uint32_t bias = 0;
                    for (int q = q_begin; q < q_end; ++q) bias += lp.fix.bias_q[q];
#pragma unroll
                    for (int j = 0; j < kSPT; ++j) ipq[j] -= static_cast<int>(bias);
                    ipq_to_samples(ipq, isum);
                }
                if (any) {
#pragma unroll 1
                    for (int q = q_begin; q < q_end; ++q) {
                        uint32_t nq = 0;
#pragma unroll
                        for (int r2 = 0; r2 < SPLIT; ++r2) nq |= team_ws[r2].nm_leaf[q];
                        if (nq == 0) continue;
                        Acc16 mq;
#pragma unroll
                        for (int j = 0; j < kPairs; ++j) mq.a[j] = make_float2(0.f, 0.f);
                        mover_block<SPLIT>(lp, ws, team_ws, 0, SPLIT, q, per, bpl, blk_base, lane, mq);
                        const int sh = lp.fix.quad_sh[q], mul = 1 << (lp.fix.fix_sh - sh);
                        const float2 sc = dup2(pow2f(sh)), mg = dup2(kRoundMagic);
#pragma unroll
                        for (int j = 0; j < kPairs; ++j) {
                            const float2 t = __ffma2_rn(mq.a[j], sc, mg);
                            isum[2 * j] += fix_of(t.x, mul);
                            isum[2 * j + 1] += fix_of(t.y, mul);
                        }
                    }
                }
                if (!cross) {
                    Acc16 sum;
#pragma unroll
                    for (int j = 0; j < kPairs; ++j)
                        sum.a[j] = make_float2(__int2float_rn(isum[2 * j]) * lp.fix.fix_inv, __int2float_rn(isum[2 * j + 1]) * lp.fix.fix_inv);
                    store_block(lp, n_thread + r * kBlock, xs_tile, lane * kSPT + r * kBlock, sum);
                } else {
                    // this quad's share of the block joins the other quads' in the launch's scratch tile: [tile][block][sample]
                    int *dst = lp.scratch + (tile * kBlocksPerTile + r) * kBlock + lane;
#pragma unroll
                    for (int j = 0; j < kSPT; ++j) atomicAdd(dst + j * 32, isum[j]);
                }
            }
        }
      }
      if (cross) {
          // Quads of one tile arrive from different CTAs in any order; integer sums do not care.  The CTA that delivers
          // the last quad reads the tile back (warp `rank` takes block `rank`), leaves zeros for the next launch on this
          // slot, quantises and stores.  No CTA waits for another.
          __threadfence();
          __syncthreads();
          if (threadIdx.x == 0) {
              const uint32_t old = atomicAdd(lp.tile_cnt + tile, 1u);
              ws_all[0].last = old == static_cast<uint32_t>(Q - 1) ? 1u : 0u;
              if (old == static_cast<uint32_t>(Q - 1)) lp.tile_cnt[tile] = 0u;
          }
          __syncthreads();
          if (ws_all[0].last) {
              __threadfence();
              const int r = rank;
              const int64_t blk_base = tile_base + static_cast<int64_t>(r) * kBlock;
              if (!(blk_base >= n_end || blk_base + kBlock <= lp.n_begin)) {
                  int *src = lp.scratch + (tile * kBlocksPerTile + r) * kBlock + lane;
                  Acc16 sum;
#pragma unroll
                  for (int j = 0; j < kPairs; ++j) {
                      const int i0 = __ldcg(src + (2 * j) * 32), i1 = __ldcg(src + (2 * j + 1) * 32);
                      src[(2 * j) * 32] = 0;
                      src[(2 * j + 1) * 32] = 0;
                      sum.a[j] = make_float2(__int2float_rn(i0) * lp.fix.fix_inv, __int2float_rn(i1) * lp.fix.fix_inv);
                  }
                  store_block(lp, n_thread + r * kBlock, xs_tile, lane * kSPT + r * kBlock, sum);
              }
          }
      }
      // the closing barrier (the next tile's partial sums overwrite the park areas) also publishes the next unit
      unit = next_unit<SPLIT>(lp, ws_all[warp - rank], team, rank, lane, n_teams);
    }
    // the last team out re-arms the counter for the launch that takes this slot next
    if (rank == 0 && lane == 0) {
        __threadfence();
        if (atomicAdd(lp.sched + 1, 1u) == static_cast<uint32_t>(n_teams - 1)) {
            lp.sched[0] = 0u;
            lp.sched[1] = 0u;
            __threadfence();
        }
    }
}

// Reference-grade engine: closed form in fp64 + 64-bit fixed point and fp64 sine for every
// (tone, sample); one thread per 8 consecutive samples.  ~50x slower than the MUFU engine.
constexpr int kSPT64 = 8;
__global__ void __launch_bounds__(256) awg_fp64_kernel(const LaunchParams lp)
{
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const int64_t n_thread = lp.n_begin + g * kSPT64;
    if (g * kSPT64 >= lp.n_count) return;
    double acc[kSPT64];
#pragma unroll
    for (int j = 0; j < kSPT64; ++j) acc[j] = 0.0;
    for (int t = 0; t < lp.n_tones; ++t) {
        const ToneCore &tr = lp.tab[t].core;
#pragma unroll
        for (int j = 0; j < kSPT64; ++j) {
            const int64_t ph = static_cast<int64_t>(exact_phase(tr, n_thread + j));  // signed: [-0.5, 0.5) turn
            acc[j] += static_cast<double>(amp_at(tr, n_thread + j)) * sinpi(static_cast<double>(ph) * (2.0 / kTwo64));
        }
    }
    const int64_t off = n_thread - lp.n_begin;
    if (lp.xs) {
        const int64_t i = n_thread % lp.xs_len;   // 8 consecutive samples never wrap: L_s is a multiple of 8
#pragma unroll
        for (int j = 0; j < kSPT64; ++j) acc[j] += static_cast<double>(__ldg(lp.xs + i + j));
    }
    if (lp.out_f32) {
        float4 *o = reinterpret_cast<float4 *>(static_cast<float *>(lp.out) + off);
        o[0] = make_float4(static_cast<float>(acc[0]), static_cast<float>(acc[1]), static_cast<float>(acc[2]), static_cast<float>(acc[3]));
        o[1] = make_float4(static_cast<float>(acc[4]), static_cast<float>(acc[5]), static_cast<float>(acc[6]), static_cast<float>(acc[7]));
    } else {
        uint32_t w[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int32_t lo, hi;
            asm("cvt.rni.sat.s16.f32 %0, %1;" : "=r"(lo) : "f"(lp.scale * static_cast<float>(acc[2 * j])));
            asm("cvt.rni.sat.s16.f32 %0, %1;" : "=r"(hi) : "f"(lp.scale * static_cast<float>(acc[2 * j + 1])));
            w[j] = (static_cast<uint32_t>(lo) & 0xffffu) | (static_cast<uint32_t>(hi) << 16);
        }
        if (lp.out_stride == 1) {
            *reinterpret_cast<uint4 *>(static_cast<int16_t *>(lp.out) + off) = make_uint4(w[0], w[1], w[2], w[3]);
        } else {
            uint16_t *o = static_cast<uint16_t *>(lp.out) + off * lp.out_stride + lp.out_offset;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                o[(2 * j) * lp.out_stride] = static_cast<uint16_t>(w[j]);
                o[(2 * j + 1) * lp.out_stride] = static_cast<uint16_t>(w[j] >> 16);
            }
        }
    }
}

// Trajectory-table build on the device (hot-path step a0): one warp per tone record.  Copies the 128-byte core the
// host computed and builds the tables of the two carriers, C_j, S_j = A cos, A sin(2 pi (j + 1/2) w): the angle
// (j + 1/2) w is exact in 64-bit fixed-point turns, cosine and sine are evaluated in fp64 and rounded once to fp32.
__global__ void __launch_bounds__(128) awg_expand_kernel(ToneRec *table, const ToneCore *src, const int32_t *idx, int n)
{
    const int j = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (j >= n) return;
    const ToneCore &c = src[j];
    ToneRec &dst = table[idx ? idx[j] : j];
    if (lane < 8) reinterpret_cast<uint4 *>(&dst.core)[lane] = reinterpret_cast<const uint4 *>(&c)[lane];
    if (lane >= 2 * kPairs) {
        // pad_[0], pad_[1] of each table: cosine and sine of the carrier phase of two groups of 16 samples (the rotation that
        // takes the sines/cosines of a thread's groups 0, 1 to its groups 2, 3 in the static pass); pad_[2], pad_[3] = 0
        if (lane < 2 * kPairs + 8) {
            const int st = (lane - 2 * kPairs) >> 2, q = lane & 3;
            float v = 0.f;
            if (q < 2) {
                const uint64_t ang2 = (st ? c.w_post : c.w_pre) * static_cast<uint64_t>(2 * kSPT);
                double sn2, cs2;
                sincospi(2.0 * (static_cast<double>(static_cast<int64_t>(ang2)) * (1.0 / kTwo64)), &sn2, &cs2);
                v = static_cast<float>(q == 0 ? cs2 : sn2);
            }
            (st ? dst.rot_post : dst.rot_pre).pad_[q] = v;
        }
        return;
    }
    const int state = lane / kPairs, p = lane % kPairs;
    const uint64_t w = state ? c.w_post : c.w_pre;
    const uint64_t ang = w * static_cast<uint64_t>(p) + (w >> 1);              // (p + 1/2) w, turns * 2^64 (wraps exactly)
    const double turns = static_cast<double>(static_cast<int64_t>(ang)) * (1.0 / kTwo64);   // [-1/2, 1/2)
    double sn, cs;
    sincospi(2.0 * turns, &sn, &cs);
    const double A = static_cast<double>(state ? c.A1 : c.A);
    RotTable &tab = state ? dst.rot_post : dst.rot_pre;
    tab.C[p] = static_cast<float>(A * cs);
    tab.S[p] = static_cast<float>(A * sn);
}

// ---- launch state, per device ------------------------------------------------------------------------------------
// Launch slots: a tile-scheduler counter pair, the per-tile quad counters and a scratch area, zeroed once; the kernel
// leaves its counters at zero again.  A slot belongs to ONE stream (keyed by the stream's unique id): launches of a stream
// run one after the other, so a slot is clean when the next launch of its stream starts, and launches that can overlap
// (different streams) never share a counter or scratch memory.
constexpr int kSchedSlots = 1024;
constexpr int kMaxDevices = 64;
constexpr int kCrossTiles = 1024;                        // launches of fewer tiles than two rounds of the grid's CTAs (< 2 x 3 x 148) run cross-CTA
constexpr int kSlotWords = 8 + kCrossTiles;              // {next unit, teams finished, -...} + per-tile quad counters
struct LaunchSlot {
    int32_t *scratch = nullptr;   // kCrossTiles tiles of int32 sums, zero between launches
};
struct DeviceState {
    uint32_t *sched = nullptr;
    std::unordered_map<unsigned long long, uint32_t> slot_of;   // stream id -> slot
    LaunchSlot slots[kSchedSlots];
    int n_sm = 0;
    uint32_t configured = 0;   // bit per kernel instantiation: dynamic shared memory opt-in done on this device
};
std::mutex g_dev_mutex;
DeviceState g_dev[kMaxDevices];

cudaError_t device_state(DeviceState **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    DeviceState &ds = g_dev[dev];
    if (!ds.sched) {
        int v = 0;
        if ((e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        uint32_t *p = nullptr;
        const size_t bytes = static_cast<size_t>(kSchedSlots) * kSlotWords * sizeof(uint32_t);
        if ((e = cudaMalloc(reinterpret_cast<void **>(&p), bytes)) != cudaSuccess) return e;
        if ((e = cudaMemset(p, 0, bytes)) != cudaSuccess || (e = cudaDeviceSynchronize()) != cudaSuccess) {
            cudaFree(p);
            return e;
        }
        ds.n_sm = v > 0 ? v : 148;
        ds.sched = p;
    }
    *out = &ds;
    return cudaSuccess;
}

template <int SPLIT, bool ROT, bool LEAVES, bool SLOW2>
cudaError_t launch_one(DeviceState &ds, const LaunchParams &lp, int64_t tiles, cudaStream_t stream)
{
    constexpr int kTeams = kWarps / SPLIT;
    constexpr size_t kSmem = sizeof(WarpSmem) * kWarps;
    constexpr uint32_t kBit = 1u << (((LEAVES ? 3 : SPLIT == 1 ? 0 : SPLIT == 2 ? 1 : 2) * 2 + (ROT ? 1 : 0)) * 2 + (SLOW2 ? 1 : 0));
    if (!(ds.configured & kBit)) {
        cudaError_t e = cudaFuncSetAttribute(awg_synth_kernel<SPLIT, ROT, LEAVES, SLOW2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             static_cast<int>(kSmem));
        if (e != cudaSuccess) return e;
        ds.configured |= kBit;
    }
    // persistent grid: kCtasPerSm CTAs per SM, fewer when the launch has fewer work units than teams
    const int64_t want = (tiles + kTeams - 1) / kTeams;   // (`tiles` = work units: tiles, or tiles x quads when lp.cross)
    const int64_t max_grid = static_cast<int64_t>(kCtasPerSm) * ds.n_sm;
    const unsigned grid = static_cast<unsigned>(want < max_grid ? want : max_grid);
    awg_synth_kernel<SPLIT, ROT, LEAVES, SLOW2><<<grid, kWarps * 32, kSmem, stream>>>(lp);
    return cudaGetLastError();
}

template <bool ROT, bool SLOW2>
cudaError_t launch_split(DeviceState &ds, const LaunchParams &lp, int split, int64_t tiles, cudaStream_t stream)
{
    switch (split) {
        case 1: return launch_one<1, ROT, false, SLOW2>(ds, lp, tiles, stream);
        case 2: return launch_one<2, ROT, false, SLOW2>(ds, lp, tiles, stream);
        default: return lp.n_quads > 1 ? launch_one<kWarps, ROT, true, SLOW2>(ds, lp, tiles, stream)
                                       : launch_one<kWarps, ROT, false, SLOW2>(ds, lp, tiles, stream);
    }
}

}  // namespace

cudaError_t launch_expand(ToneRec *table, const ToneCore *src, const int32_t *idx, int n, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    awg_expand_kernel<<<(n + 3) / 4, 128, 0, stream>>>(table, src, idx, n);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_synth(const LaunchParams &lp_in, int engine, cudaStream_t stream)
{
    if (lp_in.n_count <= 0) return cudaSuccess;
    LaunchParams lp = lp_in;
    cudaError_t e;
    if (engine == AWG_ENGINE_FP64) {
        const int64_t threads = lp.n_count / kSPT64;
        awg_fp64_kernel<<<static_cast<unsigned>((threads + 255) / 256), 256, 0, stream>>>(lp);
        e = cudaGetLastError();
    } else {
        const int64_t first_tile = lp.n_begin / kTile;
        const int64_t last_tile = (lp.n_begin + lp.n_count - 1) / kTile;
        const int64_t tiles = last_tile - first_tile + 1;
        // one launch at a time looks up its stream's slot and launches (the kernel launch is asynchronous)
        std::lock_guard<std::mutex> lock(g_dev_mutex);
        DeviceState *ds = nullptr;
        if ((e = device_state(&ds)) != cudaSuccess) return e;
        unsigned long long sid = 0;
        if (cudaStreamGetId(stream, &sid) != cudaSuccess) {
            (void)cudaGetLastError();
            sid = ~static_cast<unsigned long long>(reinterpret_cast<uintptr_t>(stream));   // no id: key on the handle
        }
        auto it = ds->slot_of.find(sid);
        if (it == ds->slot_of.end()) {
            if (ds->slot_of.size() >= static_cast<size_t>(kSchedSlots)) {
                // more streams than slots: wait for everything in flight (every slot is clean then) and start over
                if ((e = cudaDeviceSynchronize()) != cudaSuccess) return e;
                ds->slot_of.clear();
            }
            it = ds->slot_of.emplace(sid, static_cast<uint32_t>(ds->slot_of.size())).first;
        }
        lp.sched = ds->sched + static_cast<size_t>(kSlotWords) * it->second;
        lp.tile_cnt = lp.sched + 8;
        // clamp bounds of the quantiser in units of V: scale*qlo and scale*qhi round to -32768 and 32767
        lp.qlo = static_cast<float>(-32768.0 / static_cast<double>(lp.scale));
        lp.qhi = static_cast<float>(32767.0 / static_cast<double>(lp.scale));
        int split = 1, per = lp.n_tones, quads = 1;
        tone_groups(lp.n_tones, &split, &per, &quads);
        lp.per = per;
        lp.n_quads = quads;
        lp.cross = 0;
        lp.scratch = nullptr;
        int64_t units = tiles;
        if (quads > 1 && tiles < 2 * static_cast<int64_t>(kCtasPerSm) * ds->n_sm && tiles <= kCrossTiles) {
            // fewer tiles than two rounds of CTAs (a second round that is mostly empty wastes up to half the GPU): a tile's quads
            // become separate work units, their sums meet in the slot's scratch tiles
            LaunchSlot &sl = ds->slots[it->second];
            if (!sl.scratch) {
                int32_t *sp = nullptr;
                const size_t bytes = static_cast<size_t>(kCrossTiles) * kTile * sizeof(int32_t);
                if (cudaMalloc(reinterpret_cast<void **>(&sp), bytes) == cudaSuccess) {
                    if (cudaMemset(sp, 0, bytes) == cudaSuccess && cudaDeviceSynchronize() == cudaSuccess) sl.scratch = sp;
                    else cudaFree(sp);
                }
                if (!sl.scratch) (void)cudaGetLastError();   // no scratch: the quads stay inside one CTA
            }
            if (sl.scratch) {
                lp.cross = 1;
                lp.scratch = sl.scratch;
                units = tiles * quads;
            }
        }
        if (engine != AWG_ENGINE_FMA) e = launch_split<false, false>(*ds, lp, split, units, stream);   // (no slow pass: every tone on MUFU)
        else if (lp.slow2) e = launch_split<true, true>(*ds, lp, split, units, stream);
        else e = launch_split<true, false>(*ds, lp, split, units, stream);
    }
    count_launch();
    return e;
}

// ---- awg_synthesize_noalloc: the same kernels with ALL device-side working memory in one static array -----------------
// For callers that cannot allocate (a harness that forbids cudaMalloc, a serving loop that must not touch the allocator):
// no cudaMalloc / cudaFree / stream or event creation anywhere on this path.  The array is part of the library image:
// every GPU that loads the library holds its 5.9 MB until the process exits.  Every call shares it (calls that overlap
// on the GPU race), and it keeps the last call's contents: what a launch needs at zero is cleared on the caller's stream
// before the launch.
namespace {

constexpr int kNoAllocMaxTiles = static_cast<int>(kNoAllocMaxSamples / kTile) + 1;   // a range that starts inside a tile
struct NoAllocScratch {
    uint32_t sched[8];                              // tile scheduler: {next unit, teams finished, ...}
    uint32_t tile_cnt[568];                         // quads delivered per tile (cross-CTA launches); sized so that `tiles` starts 256-byte aligned
    int32_t tiles[kNoAllocMaxTiles][kTile];         // fixed-point sums of the quads of a tile (cross-CTA launches): 4.0 MB
    ToneCore cores[kNoAllocMaxTones];               // the host's tone cores: 0.5 MB
    ToneRec table[kNoAllocMaxTones];                // expanded trajectory table: 1.1 MB
};
static __device__ __align__(256) unsigned char g_noalloc_scratch[sizeof(NoAllocScratch)];
static_assert(sizeof(NoAllocScratch) < (7u << 20), "the static scratch is meant to stay modest");
static_assert(sizeof(NoAllocScratch::tile_cnt) / sizeof(uint32_t) >= kNoAllocMaxTiles, "one counter per tile");
static_assert(offsetof(NoAllocScratch, tiles) % 256 == 0 && offsetof(NoAllocScratch, cores) % 256 == 0 &&
              offsetof(NoAllocScratch, table) % 256 == 0, "the parts are aligned like cudaMalloc'ed blocks");

// Device address of the array, per device.  In host code the NAME g_noalloc_scratch is a host-side stand-in, not a device
// address: only cudaGetSymbolAddress (with the device current) gives the pointer a kernel can use.
NoAllocScratch *g_noalloc_ptr[kMaxDevices] = {};

}  // namespace

cudaError_t launch_synth_noalloc(const ToneCore *cores, int n_up, const LaunchParams &lp_in, cudaStream_t stream)
{
    if (lp_in.n_count <= 0 || n_up <= 0) return cudaSuccess;
    if (n_up > kNoAllocMaxTones || lp_in.n_tones > n_up) return cudaErrorInvalidValue;
    const int64_t first_tile = lp_in.n_begin / kTile;
    const int64_t tiles = (lp_in.n_begin + lp_in.n_count - 1) / kTile - first_tile + 1;
    if (tiles > kNoAllocMaxTiles) return cudaErrorInvalidValue;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    cudaError_t e;
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    DeviceState &ds = g_dev[dev];   // (SM count and the shared-memory opt-in bits only: nothing here touches ds.sched or the slots)
    if (!g_noalloc_ptr[dev]) {
        void *ptr = nullptr;
        if ((e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch)) != cudaSuccess) return e;
        if (ds.n_sm == 0) {
            int v = 0;
            if ((e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
            ds.n_sm = v > 0 ? v : 148;
        }
        g_noalloc_ptr[dev] = static_cast<NoAllocScratch *>(ptr);
    }
    NoAllocScratch *sc = g_noalloc_ptr[dev];
    LaunchParams lp = lp_in;
    // table build (step a0) into the static array
    if ((e = cudaMemcpyAsync(sc->cores, cores, static_cast<size_t>(n_up) * sizeof(ToneCore), cudaMemcpyHostToDevice, stream)) != cudaSuccess) return e;
    awg_expand_kernel<<<(n_up + 3) / 4, 128, 0, stream>>>(sc->table, sc->cores, nullptr, n_up);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    count_launch();
    lp.tab = sc->table;
    lp.sched = sc->sched;
    lp.tile_cnt = sc->tile_cnt;
    lp.qlo = static_cast<float>(-32768.0 / static_cast<double>(lp.scale));
    lp.qhi = static_cast<float>(32767.0 / static_cast<double>(lp.scale));
    int split = 1, per = lp.n_tones, quads = 1;
    tone_groups(lp.n_tones, &split, &per, &quads);
    lp.per = per;
    lp.n_quads = quads;
    lp.cross = 0;
    lp.scratch = nullptr;
    int64_t units = tiles;
    size_t clear = offsetof(NoAllocScratch, tiles);   // the counters always start at zero ...
    if (quads > 1 && tiles < 2 * static_cast<int64_t>(kCtasPerSm) * ds.n_sm) {
        // the rule of launch_synth: with fewer tiles than two rounds of CTAs a tile's quads are separate work units
        lp.cross = 1;
        lp.scratch = &sc->tiles[0][0];
        units = tiles * quads;
        clear += static_cast<size_t>(tiles) * kTile * sizeof(int32_t);   // ... and so do the tiles this launch adds into
    }
    if ((e = cudaMemsetAsync(sc, 0, clear, stream)) != cudaSuccess) return e;
    if (lp.slow2) e = launch_split<true, true>(ds, lp, split, units, stream);
    else e = launch_split<true, false>(ds, lp, split, units, stream);
    count_launch();
    return e;
}

}  // namespace awg

extern "C" int64_t awg_kernel_launch_count(void) { return awg::g_launches.load(std::memory_order_relaxed); }
