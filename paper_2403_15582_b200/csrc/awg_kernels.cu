// awg_kernels.cu -- sm_100a synthesis kernels: the fused WG + WC (+ quantise) of PAPER.md:158-186.
//
// Hot-path steps (SURVEY.md section 8(a) / DESIGN.md):
//   a1  per (tone, 256-sample tile) phase re-centring in 64-bit fixed point + fp64      tile_prologue()
//   a2  per tone-sample phase  c0 + c1*k (u32 turns, wraps exactly) + fp32 polynomial  mufu_loop<KIND>()
//   a3  sine: MUFU.SIN per tone-sample (MUFU engine, and every moving tile), or one MUFU.SIN + MUFU.COS per
//       8 samples rotated by a per-tone table {A cos(j w), A sin(j w)} (angle addition, static tiles of the
//       FMA engine):  A sin(phi0 + j w) = sin(phi0) * A cos(j w) + cos(phi0) * A sin(j w)        rot_loop()
//   a4  fp32 register accumulation over tones, 8 samples per thread                    acc[4] (float2)
//   a5  quantise: cvt.rni.sat.s16.f32(scale * acc)                                     store_tile()
//   a6  one 16-byte store of 8 consecutive int16 per thread                            store_tile()
// No tensor cores (north_star), no per-tone wavetable in DRAM (the paper's limiter); output
// traffic is 2 bytes per sample.
#include <cstdint>
#include <atomic>

#include "awg_internal.h"

namespace awg {

static std::atomic<int64_t> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

namespace {

constexpr int kTile = 32 * kSPT;      // samples per warp tile, anchored at absolute multiples of 256
constexpr int kHalf = kTile / 2;      // Taylor expansions are centred on the tile
constexpr int kWarps = 8;             // warps per CTA
constexpr int kBatch = 32;            // tones per prologue batch: one tone per lane
constexpr float kTurnToRad = 1.4629180792671596e-9f;   // 2*pi / 2^32: int32 phase (turns * 2^32) -> radians
constexpr double kTwo64 = 18446744073709551616.0;

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
__device__ __forceinline__ uint64_t exact_phase(const ToneRec &r, int64_t n)
{
    if ((r.cls & 0xff) == CLS_STATIC) return r.theta_pre + r.w_pre * static_cast<uint64_t>(n);
    const double u = (static_cast<double>(n) - r.ns_int) - r.ns_frac;
    if (u <= 0.0) return r.theta_pre + r.w_pre * static_cast<uint64_t>(n);
    if (u >= r.Tn) return r.theta_post + r.w_post * static_cast<uint64_t>(n);
    const double x = r.DT * profile_g(r.cls >> 8, u * r.inv_Tn);
    return r.theta_pre + r.w_pre * static_cast<uint64_t>(n) + frac_to_fix64(x);
}

// Kinds of (tone, tile) record, in the order the inner loops run them.
enum : int {
    K_NONE = -1,
    K_STATIC = 0,  // carrier only
    K_QUAD = 1,    // + k^2 term
    K_DEG4 = 2,    // + k^2..k^4
    K_DEG6 = 3,    // + k^2..k^6
    K_SBEG = 4,    // the move starts inside this tile: pre-move carrier + P(max(k - kb, 0))
    K_SEND = 5,    // the move ends inside this tile:  post-move carrier + P(max(kb - k, 0))
    K_EXACT = 6,   // anything else (both ends in one tile, T = 0, CLS_EXACT tones): fp64 per sample
    K_COUNT = 7
};

// One re-centred (tone, tile) record:
//   phase(k) = c0 + c1*k [u32 turns, wrapping] + poly(k) [radians, fp32],  k = n - tile centre
//   K_QUAD..K_DEG6: poly = k^2 (c2 + k (c3 + k (c4 + k (c5 + k c6))))     (Taylor series about the tile centre)
//   K_SBEG/K_SEND:  poly = w^2 (c2 + w^2 (c3 + w (c4 + w c5))), w = max(+-(k - kb), 0), c6 = +-kb
//   K_STATIC with the FMA engine: `rot` points at the carrier's rotation table in the tone record
struct TileRec {
    uint32_t c0, c1;
    float A;
    float c2, c3, c4, c5, c6;
    int kind;
    const float *rot;
};

// Step a1.  Lane-private: tone record `rec` at the tile whose first sample is tile_base (absolute);
// tb_d = (double)tile_base, nc = tile_base + 128.
__device__ __forceinline__ TileRec tile_prologue(const ToneRec *rec, int t, uint64_t nc, double tb_d)
{
    TileRec r;
    r.c2 = r.c3 = r.c4 = r.c5 = r.c6 = 0.f;
    r.kind = K_STATIC;
    r.rot = rec->rot_pre;
    const uint4 v0 = ldg16(rec);  // A, cls, theta_pre
    r.A = __uint_as_float(v0.x);
    const int32_t cls = static_cast<int32_t>(v0.y);
    const int c = cls & 0xff;
    const uint64_t theta_pre = u64_of(v0.z, v0.w);
    const uint4 v1 = ldg16(reinterpret_cast<const char *>(rec) + 16);  // w_pre, theta_post
    const uint64_t w_pre = u64_of(v1.x, v1.y);
    uint64_t ph, w;
    if (c == CLS_STATIC) {
        w = w_pre;
        ph = theta_pre + w * nc;
    } else {
        const uint4 v2 = ldg16(reinterpret_cast<const char *>(rec) + 32);  // w_post, ns_int
        const uint4 v3 = ldg16(reinterpret_cast<const char *>(rec) + 48);  // ns_frac, Tn
        const double Tn = f64_of(v3.z, v3.w);
        const double ua = (tb_d - f64_of(v2.z, v2.w)) - f64_of(v3.x, v3.y);  // u of the tile's first sample
        const double ub = ua + static_cast<double>(kTile - 1);
        const bool linear = (cls >> 8) == AWG_PROFILE_LINEAR;
        if (ub <= 0.0) {
            w = w_pre;
            ph = theta_pre + w * nc;
        } else if (ua >= Tn) {
            w = u64_of(v2.x, v2.y);
            ph = u64_of(v1.z, v1.w) + w * nc;
            r.rot = rec->rot_post;
        } else if (c == CLS_EXACT || (ua < 0.0 && ub > Tn)) {
            r.kind = K_EXACT;
            r.c0 = static_cast<uint32_t>(t);
            r.c1 = 0;
            return r;
        } else {
            const uint4 v4 = ldg16(reinterpret_cast<const char *>(rec) + 64);  // inv_Tn, DT
            const uint4 v5 = ldg16(reinterpret_cast<const char *>(rec) + 80);  // q1, q[0], q[1]
            const uint4 v6 = ldg16(reinterpret_cast<const char *>(rec) + 96);  // q[2], q[3], q[4]
            const double rT = f64_of(v4.x, v4.y);
            const double DT = f64_of(v4.z, v4.w);
            const float q2 = __uint_as_float(v5.z), q3 = __uint_as_float(v5.w);
            const float q4 = __uint_as_float(v6.x), q5 = __uint_as_float(v6.y), q6 = __uint_as_float(v6.z);
            if (ua >= 0.0 && ub <= Tn) {
                // whole tile inside the move (g(0) = 0 and DT g(1) = post - pre, so the closed ends are included):
                // Taylor-expand DT*g((u_c + k)/Tn) about the tile centre.  Phase and frequency (g, g') in fp64,
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
                w = w_pre + frac_to_fix64(f64_of(v5.x, v5.y) * g1);  // instantaneous frequency at the tile centre
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
                // exactly one end of the move lies inside the tile.  With w the (clamped) distance into the move
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

// Per-warp shared-memory record of one (tone, tile): 80 bytes.
//   q[0] = {c0 bits, c1 bits, A, c2};  moving kinds: q[1] = {c3, c4, c5, c6}
//   static tiles of the FMA engine:    q[1..2] = A cos(j w), j = 0..7;  q[3..4] = A sin(j w), j = 0..7
struct __align__(16) SmemRec {
    float4 q[5];
};

// Steps a2-a4, MUFU path, for `count` records starting at rec[first], all of kind KIND.  Samples go in pairs
// through the packed fp32x2 instructions of sm_100 (FMUL2 / FFMA2: one issue slot for two samples).
template <int KIND>
__device__ __forceinline__ void mufu_loop(const SmemRec *rec, int first, int count, int koff,
                                          const float2 (&kf)[kSPT / 2], const float2 (&kk)[kSPT / 2],
                                          float2 (&acc)[kSPT / 2])
{
    const float2 K2 = dup2(kTurnToRad);
#pragma unroll 2
    for (int i = first; i < first + count; ++i) {
        const float4 a = rec[i].q[0];
        const uint32_t c0 = __float_as_uint(a.x), c1 = __float_as_uint(a.y);
        const float A = a.z;
        const uint32_t base = c0 + c1 * static_cast<uint32_t>(koff);
        float4 b;
        if (KIND >= K_DEG4) b = rec[i].q[1];
#pragma unroll
        for (int j = 0; j < kSPT / 2; ++j) {
            const uint32_t p0 = base + c1 * static_cast<uint32_t>(2 * j);
            const uint32_t p1 = base + c1 * static_cast<uint32_t>(2 * j + 1);
            const float2 f = make_float2(__int2float_rn(static_cast<int32_t>(p0)), __int2float_rn(static_cast<int32_t>(p1)));
            float2 x;
            if (KIND == K_STATIC) {
                x = __fmul2_rn(f, K2);
            } else if (KIND == K_SBEG || KIND == K_SEND) {
                float2 w;
                w.x = fmaxf((KIND == K_SBEG ? kf[j].x : -kf[j].x) - b.w, 0.f);
                w.y = fmaxf((KIND == K_SBEG ? kf[j].y : -kf[j].y) - b.w, 0.f);
                const float2 w2 = __fmul2_rn(w, w);
                float2 poly = __ffma2_rn(dup2(b.z), w, dup2(b.y));
                poly = __ffma2_rn(poly, w, dup2(b.x));
                poly = __ffma2_rn(poly, w2, dup2(a.w));
                x = __ffma2_rn(f, K2, __fmul2_rn(poly, w2));
            } else {
                float2 poly;
                if (KIND == K_QUAD) {
                    poly = dup2(a.w);
                } else if (KIND == K_DEG4) {
                    poly = __ffma2_rn(dup2(b.y), kf[j], dup2(b.x));
                    poly = __ffma2_rn(poly, kf[j], dup2(a.w));
                } else {
                    poly = __ffma2_rn(dup2(b.w), kf[j], dup2(b.z));
                    poly = __ffma2_rn(poly, kf[j], dup2(b.y));
                    poly = __ffma2_rn(poly, kf[j], dup2(b.x));
                    poly = __ffma2_rn(poly, kf[j], dup2(a.w));
                }
                x = __ffma2_rn(f, K2, __fmul2_rn(poly, kk[j]));
            }
            acc[j] = __ffma2_rn(dup2(A), make_float2(mufu_sin(x.x), mufu_sin(x.y)), acc[j]);
        }
    }
}

// Steps a2-a4, angle-addition path, static tiles: per (thread, tone) ONE sine and ONE cosine of the phase at the
// thread's first sample, then 8 samples by rotation with the tone's table:
//   A sin(phi0 + j w) = sin(phi0) * [A cos(j w)] + cos(phi0) * [A sin(j w)],  j = 0..7   -> 8 FFMA2 for 8 samples.
__device__ __forceinline__ void rot_loop(const SmemRec *rec, int first, int count, int koff, float2 (&acc)[kSPT / 2])
{
#pragma unroll 2
    for (int i = first; i < first + count; ++i) {
        const float4 a = rec[i].q[0];
        const float4 c03 = rec[i].q[1], c47 = rec[i].q[2], s03 = rec[i].q[3], s47 = rec[i].q[4];
        const uint32_t p = __float_as_uint(a.x) + __float_as_uint(a.y) * static_cast<uint32_t>(koff);
        const float x = __int2float_rn(static_cast<int32_t>(p)) * kTurnToRad;
        const float2 sn = dup2(mufu_sin(x)), cs = dup2(mufu_cos(x));
        acc[0] = __ffma2_rn(sn, make_float2(c03.x, c03.y), acc[0]);
        acc[1] = __ffma2_rn(sn, make_float2(c03.z, c03.w), acc[1]);
        acc[2] = __ffma2_rn(sn, make_float2(c47.x, c47.y), acc[2]);
        acc[3] = __ffma2_rn(sn, make_float2(c47.z, c47.w), acc[3]);
        acc[0] = __ffma2_rn(cs, make_float2(s03.x, s03.y), acc[0]);
        acc[1] = __ffma2_rn(cs, make_float2(s03.z, s03.w), acc[1]);
        acc[2] = __ffma2_rn(cs, make_float2(s47.x, s47.y), acc[2]);
        acc[3] = __ffma2_rn(cs, make_float2(s47.z, s47.w), acc[3]);
    }
}

struct Acc8 {
    float v[kSPT];
};

// fp64 path for the K_EXACT records (tones whose fp32 polynomial would be inaccurate, moves shorter than
// a tile, instant retunes): exact phase per sample, same sine.
// Out of line and by value so that the hot loops keep their accumulators in registers.
__device__ __noinline__ Acc8 exact_loop(const ToneRec *tab, const SmemRec *rec, int first, int count,
                                        int64_t n_thread, Acc8 acc)
{
    for (int i = first; i < first + count; ++i) {
        const ToneRec &tr = tab[__float_as_uint(rec[i].q[0].x)];
        const float A = rec[i].q[0].z;
#pragma unroll
        for (int j = 0; j < kSPT; ++j) {
            const uint32_t p = round32(exact_phase(tr, n_thread + j));
            acc.v[j] = fmaf(A, mufu_sin(__int2float_rn(static_cast<int32_t>(p)) * kTurnToRad), acc.v[j]);
        }
    }
    return acc;
}

__device__ __forceinline__ void store_tile(const LaunchParams &lp, int64_t n_thread, const float (&acc)[kSPT])
{
    const int64_t off = n_thread - lp.n_begin;
    if (off < 0 || off >= lp.n_count) return;  // n_begin and n_count are multiples of 8: all or nothing per thread
    if (lp.out_f32) {
        float4 *o = reinterpret_cast<float4 *>(static_cast<float *>(lp.out) + off);
        o[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        o[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
    } else {
        uint32_t w[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int32_t lo, hi;
            asm("cvt.rni.sat.s16.f32 %0, %1;" : "=r"(lo) : "f"(lp.scale * acc[2 * j]));
            asm("cvt.rni.sat.s16.f32 %0, %1;" : "=r"(hi) : "f"(lp.scale * acc[2 * j + 1]));
            w[j] = (static_cast<uint32_t>(lo) & 0xffffu) | (static_cast<uint32_t>(hi) << 16);
        }
        *reinterpret_cast<uint4 *>(static_cast<int16_t *>(lp.out) + off) = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

// SPLIT warps share one 256-sample tile, each taking 1/SPLIT of the tones; a CTA holds kWarps/SPLIT tiles.
// ROT: static tiles use the angle-addition path (FMA engine) instead of one MUFU.SIN per tone-sample.
template <int SPLIT, bool ROT>
__global__ void __launch_bounds__(kWarps * 32, 4) awg_synth_kernel(const LaunchParams lp)
{
    constexpr int kTilesPerCta = kWarps / SPLIT;
    __shared__ SmemRec s_rec[kWarps][kBatch];
    __shared__ __align__(16) float s_red[SPLIT > 1 ? kWarps : 1][SPLIT > 1 ? kTile : 1];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int tile_in_cta = warp / SPLIT;
    const int rank = warp % SPLIT;

    // tiles are anchored to absolute sample indices (chunk-size invariance, SURVEY.md 8(b) "Determinism")
    const int64_t first_tile = lp.n_begin / kTile;  // n_begin >= 0
    const int64_t tile = first_tile + static_cast<int64_t>(blockIdx.x) * kTilesPerCta + tile_in_cta;
    const int64_t tile_base = tile * kTile;
    const bool tile_live = tile_base < lp.n_begin + lp.n_count;

    const int koff = lane * kSPT - kHalf;
    float2 kf[kSPT / 2], kk[kSPT / 2], acc2[kSPT / 2];
#pragma unroll
    for (int j = 0; j < kSPT / 2; ++j) {
        kf[j] = make_float2(static_cast<float>(koff + 2 * j), static_cast<float>(koff + 2 * j + 1));
        kk[j] = make_float2(kf[j].x * kf[j].x, kf[j].y * kf[j].y);
        acc2[j] = make_float2(0.f, 0.f);
    }

    const int per = (lp.n_tones + SPLIT - 1) / SPLIT;
    const int t_begin = rank * per;
    const int t_end = min(lp.n_tones, t_begin + per);
    SmemRec *rec = s_rec[warp];

    if (tile_live) {
        const uint64_t nc = static_cast<uint64_t>(tile_base + kHalf);
        const double tb_d = static_cast<double>(tile_base);
        for (int tb = t_begin; tb < t_end; tb += kBatch) {
            const int t = tb + lane;
            TileRec r;
            r.kind = K_NONE;
            if (t < t_end) r = tile_prologue(lp.tab + t, t, nc, tb_d);
            // compact the batch by kind so each inner loop is warp-uniform (no divergence)
            int n_of[K_COUNT];
            int pos = -1, before = 0;
            const unsigned lt = (1u << lane) - 1u;
#pragma unroll
            for (int kd = 0; kd < K_COUNT; ++kd) {
                const unsigned m = __ballot_sync(0xffffffffu, r.kind == kd);
                n_of[kd] = __popc(m);
                if (r.kind == kd) pos = before + __popc(m & lt);
                before += n_of[kd];
            }
            __syncwarp();  // previous batch's readers are done
            if (pos >= 0) {
                rec[pos].q[0] = make_float4(__uint_as_float(r.c0), __uint_as_float(r.c1), r.A, r.c2);
                if (ROT && r.kind == K_STATIC) {
                    const float4 *g = reinterpret_cast<const float4 *>(r.rot);
#pragma unroll
                    for (int v = 0; v < 4; ++v) rec[pos].q[1 + v] = __ldg(g + v);
                } else {
                    rec[pos].q[1] = make_float4(r.c3, r.c4, r.c5, r.c6);
                }
            }
            __syncwarp();
            int first = 0;
            if (ROT) rot_loop(rec, first, n_of[K_STATIC], koff, acc2);
            else mufu_loop<K_STATIC>(rec, first, n_of[K_STATIC], koff, kf, kk, acc2);
            first += n_of[K_STATIC];
            if (n_of[K_QUAD]) mufu_loop<K_QUAD>(rec, first, n_of[K_QUAD], koff, kf, kk, acc2);
            first += n_of[K_QUAD];
            if (n_of[K_DEG4]) mufu_loop<K_DEG4>(rec, first, n_of[K_DEG4], koff, kf, kk, acc2);
            first += n_of[K_DEG4];
            if (n_of[K_DEG6]) mufu_loop<K_DEG6>(rec, first, n_of[K_DEG6], koff, kf, kk, acc2);
            first += n_of[K_DEG6];
            if (n_of[K_SBEG]) mufu_loop<K_SBEG>(rec, first, n_of[K_SBEG], koff, kf, kk, acc2);
            first += n_of[K_SBEG];
            if (n_of[K_SEND]) mufu_loop<K_SEND>(rec, first, n_of[K_SEND], koff, kf, kk, acc2);
            first += n_of[K_SEND];
            if (n_of[K_EXACT]) {
                Acc8 a8;
#pragma unroll
                for (int j = 0; j < kSPT / 2; ++j) { a8.v[2 * j] = acc2[j].x; a8.v[2 * j + 1] = acc2[j].y; }
                a8 = exact_loop(lp.tab, rec, first, n_of[K_EXACT], tile_base + lane * kSPT, a8);
#pragma unroll
                for (int j = 0; j < kSPT / 2; ++j) acc2[j] = make_float2(a8.v[2 * j], a8.v[2 * j + 1]);
            }
        }
    }

    float acc[kSPT];
#pragma unroll
    for (int j = 0; j < kSPT / 2; ++j) { acc[2 * j] = acc2[j].x; acc[2 * j + 1] = acc2[j].y; }
    if (SPLIT > 1) {
        float4 *mine = reinterpret_cast<float4 *>(&s_red[warp][lane * kSPT]);
        mine[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        mine[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
        __syncthreads();
        if (rank != 0 || !tile_live) return;
        // fixed summation order (rank 0, 1, ...) keeps the result independent of scheduling
        for (int r2 = 1; r2 < SPLIT; ++r2) {
            const float4 *o = reinterpret_cast<const float4 *>(&s_red[warp + r2][lane * kSPT]);
            const float4 u = o[0], v = o[1];
            acc[0] += u.x; acc[1] += u.y; acc[2] += u.z; acc[3] += u.w;
            acc[4] += v.x; acc[5] += v.y; acc[6] += v.z; acc[7] += v.w;
        }
    } else if (!tile_live) {
        return;
    }
    store_tile(lp, tile_base + lane * kSPT, acc);
}

// Reference-grade engine: closed form in fp64 + 64-bit fixed point and fp64 sine for every
// (tone, sample); one thread per 8 consecutive samples.  ~50x slower than the MUFU engine.
__global__ void __launch_bounds__(256) awg_fp64_kernel(const LaunchParams lp)
{
    const int64_t g = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const int64_t n_thread = lp.n_begin + g * kSPT;
    if (g * kSPT >= lp.n_count) return;
    double acc[kSPT];
#pragma unroll
    for (int j = 0; j < kSPT; ++j) acc[j] = 0.0;
    for (int t = 0; t < lp.n_tones; ++t) {
        const ToneRec &tr = lp.tab[t];
        const double A = static_cast<double>(tr.A);
#pragma unroll
        for (int j = 0; j < kSPT; ++j) {
            const int64_t ph = static_cast<int64_t>(exact_phase(tr, n_thread + j));  // signed: [-0.5, 0.5) turn
            acc[j] += A * sinpi(static_cast<double>(ph) * (2.0 / kTwo64));
        }
    }
    float out[kSPT];
#pragma unroll
    for (int j = 0; j < kSPT; ++j) out[j] = static_cast<float>(acc[j]);
    store_tile(lp, n_thread, out);
}

// Partial trajectory-table update: one 256-byte record per block of 16 threads x 16 bytes.
__global__ void awg_scatter_kernel(ToneRec *table, const ToneRec *src, const int32_t *idx, int n)
{
    const int j = blockIdx.x;
    if (j >= n) return;
    const uint4 *s4 = reinterpret_cast<const uint4 *>(src + j);
    uint4 *d4 = reinterpret_cast<uint4 *>(table + idx[j]);
    d4[threadIdx.x] = s4[threadIdx.x];
}

template <bool ROT>
void launch_split(const LaunchParams &lp, int split, unsigned tiles, cudaStream_t stream)
{
    auto grid_for = [&](int s) { return (tiles + (kWarps / s) - 1) / (kWarps / s); };
    switch (split) {
        case 1: awg_synth_kernel<1, ROT><<<grid_for(1), kWarps * 32, 0, stream>>>(lp); break;
        case 2: awg_synth_kernel<2, ROT><<<grid_for(2), kWarps * 32, 0, stream>>>(lp); break;
        case 4: awg_synth_kernel<4, ROT><<<grid_for(4), kWarps * 32, 0, stream>>>(lp); break;
        default: awg_synth_kernel<8, ROT><<<grid_for(8), kWarps * 32, 0, stream>>>(lp); break;
    }
}

}  // namespace

cudaError_t launch_scatter(ToneRec *table, const ToneRec *src, const int32_t *idx, int n, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    awg_scatter_kernel<<<n, sizeof(ToneRec) / sizeof(uint4), 0, stream>>>(table, src, idx, n);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_synth(const LaunchParams &lp, int engine, cudaStream_t stream)
{
    if (lp.n_count <= 0) return cudaSuccess;
    if (engine == AWG_ENGINE_FP64) {
        const int64_t threads = lp.n_count / kSPT;
        awg_fp64_kernel<<<static_cast<unsigned>((threads + 255) / 256), 256, 0, stream>>>(lp);
    } else {
        const int64_t first_tile = lp.n_begin / kTile;
        const int64_t last_tile = (lp.n_begin + lp.n_count - 1) / kTile;
        const unsigned tiles = static_cast<unsigned>(last_tile - first_tile + 1);
        // Warps per tile depend on the tone count ONLY (>= 32 tones per warp, at most 8 warps), never on the
        // launch size: the order in which tone partial sums are added is then the same for every chunking,
        // which keeps the output bit-identical across chunk sizes (include/awg.h "pure function").
        int split = 1;
        while (split < kWarps && lp.n_tones / (split * 2) >= 32) split *= 2;
        if (engine == AWG_ENGINE_FMA) launch_split<true>(lp, split, tiles, stream);
        else launch_split<false>(lp, split, tiles, stream);
    }
    count_launch();
    return cudaGetLastError();
}

}  // namespace awg

extern "C" int64_t awg_kernel_launch_count(void) { return awg::g_launches.load(std::memory_order_relaxed); }
