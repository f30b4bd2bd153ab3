// awg_kernels.cu -- sm_100a synthesis kernels: the fused WG + WC (+ quantise) of PAPER.md:158-186.
//
// Hot-path steps (SURVEY.md section 8(a) / DESIGN.md):
//   a1  per (tone, 256-sample tile) phase re-centring in 64-bit fixed point + fp64      tile_prologue()
//   a2  per tone-sample phase  c0 + c1*k (u32 turns, wraps exactly) + fp32 polynomial  tone_loop<DEG>()
//   a3  sin through MUFU.SIN (sin.approx.ftz.f32)                                      mufu_sin()
//   a4  fp32 register accumulation over tones, 8 samples per thread                    acc[8]
//   a5  quantise: cvt.rni.sat.s16.f32(scale * acc)                                     store_tile()
//   a6  one 16-byte store of 8 consecutive int16 per thread                            store_tile()
// The engine is XU(MUFU)-bound by design: no tensor cores (this is not a dense contraction), no
// per-tone wavetable in DRAM (the paper's limiter), output traffic 2 bytes/sample.
#include <cstdint>
#include <atomic>

#include "awg_internal.h"

namespace awg {

static std::atomic<int64_t> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

namespace {

constexpr int kSPT = 8;               // consecutive samples per thread -> one 16-byte int16 store
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

// g(s) of the move profile: phase gained over the carrier is DT*g(s) cycles.
__device__ __forceinline__ double profile_g(int profile, double s)
{
    if (profile == AWG_PROFILE_LINEAR) return 0.5 * s * s;
    double s2 = s * s;
    return s2 * s2 * (2.5 + s * (s - 3.0));  // 5/2 s^4 - 3 s^5 + s^6   (Eq. 10 p(i), prefactor T: G1)
}

// Exact (fp64 + 64-bit fixed point) phase of tone t at absolute sample n, in turns * 2^64.
__device__ __forceinline__ uint64_t exact_phase(const ToneTable &T, int t, int64_t n)
{
    const int32_t cls = T.cls[t];
    if ((cls & 0xff) == CLS_STATIC) return T.theta_pre[t] + T.w_pre[t] * static_cast<uint64_t>(n);
    const double u = static_cast<double>(n - T.ns_int[t]) - T.ns_frac[t];
    const double Tn = T.Tn[t];
    if (u <= 0.0) return T.theta_pre[t] + T.w_pre[t] * static_cast<uint64_t>(n);
    if (u >= Tn) return T.theta_post[t] + T.w_post[t] * static_cast<uint64_t>(n);
    const double x = T.DT[t] * profile_g(cls >> 8, u * T.inv_Tn[t]);
    return T.theta_pre[t] + T.w_pre[t] * static_cast<uint64_t>(n) + frac_to_fix64(x);
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
struct TileRec {
    uint32_t c0, c1;
    float A;
    float c2, c3, c4, c5, c6;
    int kind;
};

// Step a1.  Lane-private: tone t at the tile whose first sample is tile_base (absolute).
__device__ __forceinline__ TileRec tile_prologue(const ToneTable &T, int t, int64_t tile_base)
{
    TileRec r;
    r.c2 = r.c3 = r.c4 = r.c5 = r.c6 = 0.f;
    r.A = T.A[t];
    const int32_t cls = T.cls[t];
    const int c = cls & 0xff;
    const uint64_t nc = static_cast<uint64_t>(tile_base + kHalf);
    const double two_pi = 6.283185307179586476925286766559;
    uint64_t ph, w;
    r.kind = K_STATIC;
    if (c == CLS_STATIC) {
        w = T.w_pre[t];
        ph = T.theta_pre[t] + w * nc;
    } else {
        const double Tn = T.Tn[t];
        const double ua = static_cast<double>(tile_base - T.ns_int[t]) - T.ns_frac[t];  // u of the tile's first sample
        const double ub = ua + static_cast<double>(kTile - 1);
        const bool linear = (cls >> 8) == AWG_PROFILE_LINEAR;
        if (ub <= 0.0) {
            w = T.w_pre[t];
            ph = T.theta_pre[t] + w * nc;
        } else if (ua >= Tn) {
            w = T.w_post[t];
            ph = T.theta_post[t] + w * nc;
        } else if (c == CLS_EXACT || (ua < 0.0 && ub > Tn)) {
            r.kind = K_EXACT;
            r.c0 = static_cast<uint32_t>(t);
            r.c1 = 0;
            return r;
        } else if (ua >= 0.0 && ub <= Tn) {
            // whole tile inside the move (g(0) = 0 and DT g(1) = post - pre, so the closed ends are included):
            // Taylor-expand DT*g((u_c + k)/Tn) about the tile centre
            const double rT = T.inv_Tn[t];
            const double s = (ua + static_cast<double>(kHalf)) * rT;
            const double DT = T.DT[t];
            double g0, g1, g2, g3 = 0.0, g4 = 0.0, g5 = 0.0, g6 = 0.0;
            if (linear) {
                g0 = 0.5 * s * s; g1 = s; g2 = 1.0;
            } else {
                const double s2 = s * s;
                g0 = s2 * s2 * (2.5 + s * (s - 3.0));
                g1 = s2 * s * (10.0 + s * (6.0 * s - 15.0));
                g2 = s2 * (30.0 + s * (30.0 * s - 60.0));
                g3 = s * (60.0 + s * (120.0 * s - 180.0));
                g4 = 60.0 + s * (360.0 * s - 360.0);
                g5 = 720.0 * s - 360.0;
                g6 = 720.0;
            }
            w = T.w_pre[t];
            ph = T.theta_pre[t] + w * nc + frac_to_fix64(DT * g0);
            double q = DT * rT;                       // (f1-f0)/fs, cycles per sample
            w += frac_to_fix64(q * g1);               // instantaneous frequency at the tile centre
            q *= rT * two_pi;  r.c2 = static_cast<float>(q * g2 * 0.5);
            r.kind = K_QUAD;
            if (c >= CLS_DEG4) {
                q *= rT;  r.c3 = static_cast<float>(q * g3 * (1.0 / 6.0));
                q *= rT;  r.c4 = static_cast<float>(q * g4 * (1.0 / 24.0));
                r.kind = K_DEG4;
                if (c >= CLS_DEG6) {
                    q *= rT;  r.c5 = static_cast<float>(q * g5 * (1.0 / 120.0));
                    q *= rT;  r.c6 = static_cast<float>(q * g6 * (1.0 / 720.0));
                    r.kind = K_DEG6;
                }
            }
        } else {
            // exactly one end of the move lies inside the tile.  With w the (clamped) distance into the move
            // from that end, both ends have the same polynomial: DT (w/Tn)^2/2 (LINEAR) or
            // DT (5/2 (w/Tn)^4 - 3 (w/Tn)^5 + (w/Tn)^6) (MINJERK) on top of the carrier valid outside the move
            // [at the end: g(1+x) - (1/2 + x) = 5/2 x^4 + 3 x^5 + x^6, x = -w/Tn].
            const double rT = T.inv_Tn[t];
            const double DT = T.DT[t] * two_pi;
            const double r2 = rT * rT;
            if (linear) {
                r.c2 = static_cast<float>(0.5 * DT * r2);
            } else {
                r.c3 = static_cast<float>(2.5 * DT * r2 * r2);
                r.c4 = static_cast<float>(-3.0 * DT * r2 * r2 * rT);
                r.c5 = static_cast<float>(DT * r2 * r2 * r2);
            }
            if (ua < 0.0) {   // start inside: u = 0 at k = kb
                r.kind = K_SBEG;
                r.c6 = static_cast<float>(-(ua + static_cast<double>(kHalf)));
                w = T.w_pre[t];
                ph = T.theta_pre[t] + w * nc;
            } else {          // end inside: u = Tn at k = kb; stored negated (w = max(kb - k, 0) = max(-k - (-kb), 0))
                r.kind = K_SEND;
                r.c6 = static_cast<float>(-(Tn - ua - static_cast<double>(kHalf)));
                w = T.w_post[t];
                ph = T.theta_post[t] + w * nc;
            }
        }
    }
    r.c0 = round32(ph);
    r.c1 = round32(w);
    return r;
}

struct __align__(16) SmemRec {
    float4 a;  // {c0 bits, c1 bits, A, c2}
    float4 b;  // {c3, c4, c5, c6}
};

// Steps a2-a4 for `count` records starting at rec[first], all of kind KIND.
template <int KIND>
__device__ __forceinline__ void tone_loop(const SmemRec *rec, int first, int count, int koff,
                                          const float (&kf)[kSPT], const float (&kk)[kSPT], float (&acc)[kSPT])
{
#pragma unroll 2
    for (int i = first; i < first + count; ++i) {
        const float4 a = rec[i].a;
        const uint32_t c0 = __float_as_uint(a.x), c1 = __float_as_uint(a.y);
        const float A = a.z;
        const uint32_t base = c0 + c1 * static_cast<uint32_t>(koff);
        float4 b;
        if (KIND >= K_DEG4) b = rec[i].b;
#pragma unroll
        for (int j = 0; j < kSPT; ++j) {
            const uint32_t p = base + c1 * static_cast<uint32_t>(j);
            const float f = __int2float_rn(static_cast<int32_t>(p));
            float x;
            if (KIND == K_STATIC) {
                x = f * kTurnToRad;
            } else if (KIND == K_SBEG || KIND == K_SEND) {
                const float w = fmaxf((KIND == K_SBEG ? kf[j] : -kf[j]) - b.w, 0.f);
                const float w2 = w * w;
                const float poly = fmaf(fmaf(fmaf(b.z, w, b.y), w, b.x), w2, a.w);
                x = fmaf(f, kTurnToRad, poly * w2);
            } else {
                float poly;
                if (KIND == K_QUAD) poly = a.w;
                else if (KIND == K_DEG4) poly = fmaf(fmaf(b.y, kf[j], b.x), kf[j], a.w);
                else poly = fmaf(fmaf(fmaf(fmaf(b.w, kf[j], b.z), kf[j], b.y), kf[j], b.x), kf[j], a.w);
                x = fmaf(f, kTurnToRad, poly * kk[j]);
            }
            acc[j] = fmaf(A, mufu_sin(x), acc[j]);
        }
    }
}

struct Acc8 {
    float v[kSPT];
};

// fp64 path for the K_EXACT records (tones whose fp32 polynomial would be inaccurate, moves shorter than
// a tile, instant retunes): exact phase per sample, same sine.
// Out of line and by value so that the hot loops keep their accumulators in registers.
__device__ __noinline__ Acc8 exact_loop(const ToneTable &T, const SmemRec *rec, int first, int count,
                                        int64_t n_thread, Acc8 acc)
{
    for (int i = first; i < first + count; ++i) {
        const int t = static_cast<int>(__float_as_uint(rec[i].a.x));
        const float A = rec[i].a.z;
#pragma unroll
        for (int j = 0; j < kSPT; ++j) {
            const uint32_t p = round32(exact_phase(T, t, n_thread + j));
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
template <int SPLIT>
__global__ void __launch_bounds__(kWarps * 32) awg_mufu_kernel(const LaunchParams lp)
{
    constexpr int kTilesPerCta = kWarps / SPLIT;
    __shared__ SmemRec s_rec[kWarps][kBatch];
    __shared__ __align__(16) float s_red[SPLIT > 1 ? kWarps : 1][SPLIT > 1 ? kTile : 1];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int tile_in_cta = warp / SPLIT;
    const int rank = warp % SPLIT;
    const ToneTable &T = lp.tab;

    // tiles are anchored to absolute sample indices (chunk-size invariance, SURVEY.md 8(b) "Determinism")
    const int64_t first_tile = lp.n_begin / kTile;  // n_begin >= 0
    const int64_t tile = first_tile + static_cast<int64_t>(blockIdx.x) * kTilesPerCta + tile_in_cta;
    const int64_t tile_base = tile * kTile;
    const bool tile_live = tile_base < lp.n_begin + lp.n_count;

    const int koff = lane * kSPT - kHalf;
    float kf[kSPT], kk[kSPT], acc[kSPT];
#pragma unroll
    for (int j = 0; j < kSPT; ++j) {
        kf[j] = static_cast<float>(koff + j);
        kk[j] = kf[j] * kf[j];
        acc[j] = 0.f;
    }

    const int per = (T.n_tones + SPLIT - 1) / SPLIT;
    const int t_begin = rank * per;
    const int t_end = min(T.n_tones, t_begin + per);
    SmemRec *rec = s_rec[warp];

    if (tile_live) {
        for (int tb = t_begin; tb < t_end; tb += kBatch) {
            const int t = tb + lane;
            TileRec r;
            r.kind = K_NONE;
            if (t < t_end) r = tile_prologue(T, t, tile_base);
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
                rec[pos].a = make_float4(__uint_as_float(r.c0), __uint_as_float(r.c1), r.A, r.c2);
                rec[pos].b = make_float4(r.c3, r.c4, r.c5, r.c6);
            }
            __syncwarp();
            int first = 0;
            tone_loop<K_STATIC>(rec, first, n_of[K_STATIC], koff, kf, kk, acc);  first += n_of[K_STATIC];
            if (n_of[K_QUAD]) tone_loop<K_QUAD>(rec, first, n_of[K_QUAD], koff, kf, kk, acc);
            first += n_of[K_QUAD];
            if (n_of[K_DEG4]) tone_loop<K_DEG4>(rec, first, n_of[K_DEG4], koff, kf, kk, acc);
            first += n_of[K_DEG4];
            if (n_of[K_DEG6]) tone_loop<K_DEG6>(rec, first, n_of[K_DEG6], koff, kf, kk, acc);
            first += n_of[K_DEG6];
            if (n_of[K_SBEG]) tone_loop<K_SBEG>(rec, first, n_of[K_SBEG], koff, kf, kk, acc);
            first += n_of[K_SBEG];
            if (n_of[K_SEND]) tone_loop<K_SEND>(rec, first, n_of[K_SEND], koff, kf, kk, acc);
            first += n_of[K_SEND];
            if (n_of[K_EXACT]) {
                Acc8 a8;
#pragma unroll
                for (int j = 0; j < kSPT; ++j) a8.v[j] = acc[j];
                a8 = exact_loop(T, rec, first, n_of[K_EXACT], tile_base + lane * kSPT, a8);
#pragma unroll
                for (int j = 0; j < kSPT; ++j) acc[j] = a8.v[j];
            }
        }
    }

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
    const ToneTable &T = lp.tab;
    double acc[kSPT];
#pragma unroll
    for (int j = 0; j < kSPT; ++j) acc[j] = 0.0;
    for (int t = 0; t < T.n_tones; ++t) {
        const double A = static_cast<double>(T.A[t]);
#pragma unroll
        for (int j = 0; j < kSPT; ++j) {
            const int64_t ph = static_cast<int64_t>(exact_phase(T, t, n_thread + j));  // signed: [-0.5, 0.5) turn
            acc[j] += A * sinpi(static_cast<double>(ph) * (2.0 / kTwo64));
        }
    }
    float out[kSPT];
#pragma unroll
    for (int j = 0; j < kSPT; ++j) out[j] = static_cast<float>(acc[j]);
    store_tile(lp, n_thread, out);
}

}  // namespace

cudaError_t launch_mufu(const LaunchParams &lp, cudaStream_t stream)
{
    if (lp.n_count <= 0) return cudaSuccess;
    const int64_t first_tile = lp.n_begin / kTile;
    const int64_t last_tile = (lp.n_begin + lp.n_count - 1) / kTile;
    const int64_t tiles = last_tile - first_tile + 1;
    // Warps per tile depend on the tone count ONLY (>= 32 tones per warp, at most 8 warps), never on the
    // launch size: the order in which tone partial sums are added is then the same for every chunking,
    // which keeps the output bit-identical across chunk sizes (include/awg.h "pure function").
    const int N = lp.tab.n_tones;
    int split = 1;
    while (split < kWarps && N / (split * 2) >= 32) split *= 2;
    auto grid_for = [&](int s) { return static_cast<unsigned>((tiles + (kWarps / s) - 1) / (kWarps / s)); };
    switch (split) {
        case 1: awg_mufu_kernel<1><<<grid_for(1), kWarps * 32, 0, stream>>>(lp); break;
        case 2: awg_mufu_kernel<2><<<grid_for(2), kWarps * 32, 0, stream>>>(lp); break;
        case 4: awg_mufu_kernel<4><<<grid_for(4), kWarps * 32, 0, stream>>>(lp); break;
        default: awg_mufu_kernel<8><<<grid_for(8), kWarps * 32, 0, stream>>>(lp); break;
    }
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_fp64(const LaunchParams &lp, cudaStream_t stream)
{
    if (lp.n_count <= 0) return cudaSuccess;
    const int64_t threads = lp.n_count / kSPT;
    const unsigned grid = static_cast<unsigned>((threads + 255) / 256);
    awg_fp64_kernel<<<grid, 256, 0, stream>>>(lp);
    count_launch();
    return cudaGetLastError();
}

}  // namespace awg

extern "C" int64_t awg_kernel_launch_count(void) { return awg::g_launches.load(std::memory_order_relaxed); }
