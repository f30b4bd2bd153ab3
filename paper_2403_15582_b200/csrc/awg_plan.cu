// awg_plan.cu -- host side of the C ABI: plan, trajectory table (hot-path step a0), synthesis entry points.
//
// The trajectory table is kept on the host in x87 long double / 64-bit fixed point; the host uploads one 128-byte
// core per tone (carriers, move window, move polynomial) and a device kernel expands it into the 384-byte record of
// awg_internal.h (it builds the pair tables of the angle-addition engine).  Carrier phases are unsigned 64-bit fixed-point
// turns, so theta + w*n is exact mod 1 for any absolute sample index n: this is the modf of Eq. 14
// done in integers, and it is what keeps 35 ms x 560 MS/s (5.6e6 cycles) and 1 s x
// 100 MS/s (1e8 cycles) phases at full precision.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <functional>
#include <limits>
#include <mutex>
#include <new>
#include <thread>
#include <utility>
#include <vector>

#include "awg_internal.h"
#include "awg_plan.h"

namespace awg {

thread_local char g_err[512] = "";

// Host loops over tones (x87 long double planning and table cores, 0.1 - 0.5 us per tone) run on a few threads once they are
// long: body(begin, end) touches only the tones of its own range, and every tone goes through the same arithmetic whichever
// thread takes it.  The threads live for one call (creating one costs about 15 us: `grain` = the shortest range worth one,
// 512 tones of trajectory planning, 1024 tone cores; at most 8 threads).
constexpr int kThreadedFrom = 2048;   // tones per call from which the planning loops are threaded (below: the plain loop)

template <class Body>
static void parallel_tones(int n, int grain, Body body)
{
    constexpr int kMaxThreads = 8;
    static const int hw = static_cast<int>(std::thread::hardware_concurrency());   // (reads /sys: 20 us per call)
    const int nt = std::min(std::min(kMaxThreads, hw > 0 ? hw : 1), n / grain);
    if (nt <= 1) {
        body(0, n);
        return;
    }
    const int per = (n + nt - 1) / nt;
    std::vector<std::thread> helpers;
    helpers.reserve(static_cast<size_t>(nt - 1));
    int done = per;   // [0, per) is the caller's own range; ranges from `done` on still have no thread
    try {
        for (int t = 1; t < nt && t * per < n; ++t) {
            const int b = t * per, e = std::min(n, b + per);
            helpers.emplace_back([body, b, e] { body(b, e); });
            done = e;
        }
    } catch (...) {
        // no more threads to be had: the caller takes the rest itself
    }
    body(0, std::min(n, per));
    if (done < n) body(done, n);
    for (std::thread &h : helpers) h.join();
}

awg_status fail(awg_status code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

awg_status fail_cuda(cudaError_t e, const char *what)
{
    return fail(AWG_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

namespace {

const long double kTwoPiL = 6.283185307179586476925286766559005768L;
constexpr int kRadius = kBlock / 2;  // half of the 512-sample block (span of one Taylor re-centring)

// frac(x) as 64-bit fixed-point turns.
uint64_t frac64(long double x)
{
    long double fr;                        // x - floor(x) in [0, 1], rounded once
    if (fabsl(x) < 9.0e18L) {
        fr = x - static_cast<long double>(static_cast<int64_t>(x));   // exact; in (-1, 1)  (no libm call on the table-build path)
        if (fr < 0.0L) fr += 1.0L;
    } else {
        fr = x - floorl(x);
    }
    const long double v = fr * 18446744073709551616.0L;   // [0, 2^64], exact
    if (!(v < 18446744073709551616.0L)) return 0;  // rounded up to one full turn
    return static_cast<uint64_t>(v);
}

bool finite_all(const double *a, int n)
{
    for (int i = 0; i < n; ++i)
        if (!std::isfinite(a[i])) return false;
    return true;
}

// Polynomial class of a moving tone (which Taylor terms of DT*g(s) matter inside a 512-sample block).
int classify(int profile, long double DT, long double Tn)
{
    if (!(Tn >= 2.0L * kRadius)) return CLS_EXACT;  // move shorter than a tile: every tile straddles anyway
    const double a = static_cast<double>(fabsl(DT) / Tn);  // |f1-f0|/fs, cycles per sample
    const double r = static_cast<double>(1.0L / Tn);
    const double R = kRadius;
    const double tol_drop = 2e-8;   // cycles: dropped Taylor terms
    const double max_mag = 0.25;    // cycles: fp32 polynomial magnitude (its rounding error is ~2^-23 of this)
    // blocks that contain one end of the move evaluate DT*g over up to 2R samples from that end in fp32
    const double sg = 2.0 * R * r;
    const double DTa = static_cast<double>(fabsl(DT));
    if (profile == AWG_PROFILE_LINEAR) {
        const double t2 = a * r * 0.5 * R * R;
        return (t2 <= max_mag && DTa * 0.5 * sg * sg <= 4.0 * max_mag) ? CLS_QUAD : CLS_EXACT;
    }
    if (DTa * sg * sg * sg * sg * (2.5 + 3.0 * sg + sg * sg) > max_mag) return CLS_EXACT;
    // sup |g^(m)| on [0,1] for g = 5/2 s^4 - 3 s^5 + s^6: 1.875, 5.7735, 60, 360, 720
    const double t2 = a * r * (1.875 / 2.0) * R * R;
    const double t3 = a * r * r * (5.7735 / 6.0) * R * R * R;
    const double t4 = a * r * r * r * (60.0 / 24.0) * R * R * R * R;
    const double t5 = a * r * r * r * r * (360.0 / 120.0) * R * R * R * R * R;
    const double t6 = a * r * r * r * r * r * R * R * R * R * R * R;
    if (t2 + t3 + t4 + t5 + t6 > max_mag) return CLS_EXACT;
    if (t3 + t4 + t5 + t6 <= tol_drop) return CLS_QUAD;
    if (t5 + t6 <= tol_drop) return CLS_DEG4;
    return CLS_DEG6;
}

// Polynomial class of an exponential chirp f = f0 e^(L s), s = u/Tn (G20).  The k-th derivative of the phase with
// respect to the sample index is (f/fs) a^(k-1) cycles per sample^k with a = L/Tn, so the Taylor terms about a block centre
// are t_k = f_max/fs a^(k-1) R^k / k! at the block's edge; the kernel carries terms up to k = 6 (block_prologue()).
int classify_exp(long double f0, long double f1, long double fs, long double L, long double Tn)
{
    if (!(Tn >= 2.0L * kRadius)) return CLS_EXACT;
    const double R = kRadius;
    const double x = static_cast<double>(fabsl(L) / Tn) * R;                       // a R
    const double fm = static_cast<double>(std::max(fabsl(f0), fabsl(f1)) / fs);    // cycles per sample
    if (!(x < 0.5)) return CLS_EXACT;
    double t[9];
    t[1] = fm * R;
    for (int k = 2; k <= 8; ++k) t[k] = t[k - 1] * x / k;
    const double rest = t[7] + t[8] / (1.0 - x / 9.0);   // everything beyond the sixth term (the series falls faster than x/9 per term)
    const double tol_drop = 2e-8, max_mag = 0.25;         // as in classify()
    if (rest > tol_drop || t[2] + t[3] + t[4] + t[5] + t[6] > max_mag) return CLS_EXACT;
    // the block that holds one end of the move: the same series counted from that end, up to 2R samples into the move, kept
    // up to the fourth power (K_XEDGE)
    const double x2 = 2.0 * x;
    double e[6];
    e[1] = fm * 2.0 * R;
    for (int k = 2; k <= 5; ++k) e[k] = e[k - 1] * x2 / k;
    if (e[5] / (1.0 - x2 / 6.0) > tol_drop || e[2] + e[3] + e[4] > 4.0 * max_mag) return CLS_EXACT;
    if (t[3] + t[4] + t[5] + t[6] + rest <= tol_drop) return CLS_QUAD;
    if (t[5] + t[6] + rest <= tol_drop) return CLS_DEG4;
    return CLS_DEG6;
}

// Slow movers (flag CLS_SLOW_FLAG): inside its move the tone changes frequency so slowly that, over a whole tile, the
// angle-addition engine can carry it: a cubic phase polynomial about the tile centre gives the phase at the pair centres
// of a thread's four groups of 16 samples, and the pair tables (built at the tile-centre frequency) are moved to the
// frequency at the thread's own centre by a first-order correction (kernel: slow pass).  Bounds with
// R = kTile/2 (half a tile), h = 7.5 (half a group), g = 24 (distance of the outer groups' centres from the thread's
// centre), Taylor coefficients C_m = a r^(m-1) sup|g^(m)| / m! in turns per sample^m (sup|g^(m)| on [0,1] for the
// minimum-jerk g: 1.875, 5.7735, 60, 360, 720 for m = 2..6):
//   dropped phase terms  C4 R^4 + C5 R^5 + C6 R^6            <= 2e-8 turn
//   dropped frequency    (4 C4 R^3 + 5 C5 R^4 + 6 C6 R^5) h  <= 2e-8 turn
//   frequency drift between the centre the tables are corrected for and a group's centre  (2 C2 + 6 C3 R) g h <= 4e-7 turn
//     (g = 24 with one correction per thread; tones that fail it but pass with g = 8 get one correction per pair of groups)
//   curvature inside a group  (C2 + 3 C3 R + 6 C4 R^2) h^2   <= 3e-7 turn
//   second order of the table correction  (2 pi h (2 C2 R + 3 C3 R^2))^2 / 2 <= 2e-7
//   fp32 polynomial magnitude  C2 R^2 + C3 R^3 <= 0.25 turn
// Returns 0 (not a slow mover), 1 (one table correction per thread: 1.25 multiply-adds per tone-sample) or 2 (the drift bound
// holds only with one correction per pair of groups, g = 8: 1.5 multiply-adds per tone-sample).
int is_slow_mover(int profile, long double DT, long double Tn)
{
    if (!(Tn >= 2.0L * kTile)) return 0;
    const double a = static_cast<double>(fabsl(DT) / Tn), r = static_cast<double>(1.0L / Tn);
    const double R = kTile / 2, h = 0.5 * (kSPT - 1);
    const bool lin = profile == AWG_PROFILE_LINEAR;
    const double C2 = a * r * (lin ? 1.0 : 1.875) / 2.0;
    const double C3 = lin ? 0.0 : a * r * r * 5.7735 / 6.0;
    const double C4 = lin ? 0.0 : a * r * r * r * 60.0 / 24.0;
    const double C5 = lin ? 0.0 : a * r * r * r * r * 360.0 / 120.0;
    const double C6 = lin ? 0.0 : a * r * r * r * r * r;
    const double R2 = R * R, R3 = R2 * R, R4 = R3 * R, R5 = R4 * R, R6 = R5 * R;
    if (C4 * R4 + C5 * R5 + C6 * R6 > 2e-8) return 0;
    if ((4.0 * C4 * R3 + 5.0 * C5 * R4 + 6.0 * C6 * R5) * h > 2e-8) return 0;
    int tables = 1;
    if ((2.0 * C2 + 6.0 * C3 * R) * (1.5 * kSPT) * h > 4e-7) {
        if ((2.0 * C2 + 6.0 * C3 * R) * (0.5 * kSPT) * h > 4e-7) return 0;
        tables = 2;
    }
    if ((C2 + 3.0 * C3 * R + 6.0 * C4 * R2) * h * h > 3e-7) return 0;
    const double x = 6.283185307179586 * h * (2.0 * C2 * R + 3.0 * C3 * R2);
    if (0.5 * x * x > 2e-7) return 0;
    return C2 * R2 + C3 * R3 <= 0.25 ? tables : 0;
}

void make_static(HostTone &h)
{
    h.profile = AWG_PROFILE_STATIC;
    h.cls = CLS_STATIC;
    h.f1 = h.f0;
    h.ns_int = 0;
    h.ns_frac = 0.0;
    h.Tn = 0.0L;
    h.T = 0.0L;
    h.DT = 0.0L;
    h.theta_post = h.theta_pre;
    h.w_post = h.w_pre;
}

// Fills the move part of h (everything but theta_pre/w_pre/f0/A) for a move f0 -> f1 that starts at the
// real sample position ns = ns_int + ns_frac and lasts T seconds.  `f_delta_ts` = (f1-f0)*t_start in cycles.
void make_move(HostTone &h, long double fs, long double f1, int profile, long double T, int64_t ns_int,
               double ns_frac, long double delta_times_tstart)
{
    const long double D = f1 - h.f0;
    if (profile == AWG_PROFILE_STATIC || D == 0.0L) {
        make_static(h);
        return;
    }
    h.profile = profile;
    h.f1 = f1;
    h.T = T;
    h.Tn = T * fs;
    h.ns_int = ns_int;
    h.ns_frac = ns_frac;
    h.DT = D * T;
    h.w_post = frac64(f1 / fs);
    // after the move: Phi = theta + f0 t_s + f1 (t - t_s) + T (f0 - f1)/2   (Eq. 10 branch 2)
    //                     = [theta - (f1-f0) t_s - DT/2] + (f1/fs) n
    h.theta_post = h.theta_pre - frac64(delta_times_tstart) - frac64(h.DT / 2.0L);
    h.expL = 0.0L;
    if (profile == AWG_PROFILE_EXP) {
        // Exponential chirp (G20): f = f0 r^s, r = f1/f0; cycles over the whole move = DT / ln r, so after it
        //   Phi = [theta - (f1-f0) t_s - (f1 T - DT/ln r)] + (f1/fs) n.
        h.expL = log1pl(D / h.f0);
        h.theta_post = h.theta_pre - frac64(delta_times_tstart) - frac64(f1 * T - h.DT / h.expL);
        // blocks wholly inside the move take the MUFU pass with a Taylor polynomial about the block centre, the blocks that hold
        // the start or the end of the move a power series from that end (classify_exp)
        h.cls = classify_exp(h.f0, f1, fs, h.expL, h.Tn);
        return;
    }
    h.cls = classify(profile, h.DT, h.Tn);
    if (h.cls != CLS_EXACT) {
        const int slow = is_slow_mover(profile, h.DT, h.Tn);
        if (slow >= 1) h.cls |= CLS_SLOW_FLAG;
        if (slow == 2) h.cls |= CLS_SLOW2_FLAG;
    }
}

long double profile_h(int profile, long double s)  // frequency ramp 0 -> 1
{
    if (profile == AWG_PROFILE_LINEAR) return s;
    return s * s * s * (10.0L + s * (6.0L * s - 15.0L));
}

long double profile_g(int profile, long double s)  // its integral
{
    if (profile == AWG_PROFILE_LINEAR) return 0.5L * s * s;
    return s * s * s * s * (2.5L + s * (s - 3.0L));
}

}  // namespace

// ---- device table versions ---------------------------------------------------------------------

static void fill_core(const HostTone &h, ToneCore &r)
{
    std::memset(&r, 0, sizeof r);
    r.A = h.A;
    r.cls = (h.profile << 8) | h.cls;
    r.A1 = h.A;
    if (h.amp_prof != AWG_PROFILE_STATIC) {
        r.cls |= CLS_AMP_FLAG;
        r.A1 = h.A1;
        r.amp_ns = static_cast<double>(h.amp_ns);
        r.amp_Tn = static_cast<float>(h.amp_Tn);
        r.amp_prof = h.amp_prof;
    }
    r.theta_pre = h.theta_pre;
    r.w_pre = h.w_pre;
    r.theta_post = h.theta_post;
    r.w_post = h.w_post;
    r.ns_int = static_cast<double>(h.ns_int);
    r.ns_frac = h.ns_frac;
    r.Tn = static_cast<double>(h.Tn);
    if (h.Tn > 0.0L) {
        const long double rT = 1.0L / h.Tn;
        r.inv_Tn = static_cast<double>(rT);
        r.DT = static_cast<double>(h.DT);
        r.q1 = static_cast<double>(h.DT * rT);
        // 2 pi DT / Tn^k / k!, k = 2..6, for fp32 consumers: double arithmetic is ample (and far cheaper than x87 here)
        static const double inv_fact[5] = {1.0 / 2.0, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0, 1.0 / 720.0};
        const double rTd = r.inv_Tn;
        double q = 6.283185307179586476925286766559 * r.q1;
        for (int k = 2; k <= 6; ++k) {
            q *= rTd;
            r.q[k - 2] = static_cast<float>(q * inv_fact[k - 2]);
        }
        if (h.profile == AWG_PROFILE_EXP) {
            // exponential chirp: its Taylor coefficients are a geometric sequence built in block_prologue(); q[0..3] carry
            // f0 T (cycles) and ln(f1/f0) as two doubles instead of the five scales
            const double F = static_cast<double>(h.f0 * h.T), Lr = static_cast<double>(h.expL);
            std::memcpy(&r.q[0], &F, sizeof F);
            std::memcpy(&r.q[2], &Lr, sizeof Lr);
        }
    }
}

// Makes the device table current on `stream`.  A changed table goes to the next of kTableVersions device
// copies, so kernels still reading the previous version are never disturbed.  The host uploads 128-byte tone cores
// and the expand kernel builds the records (with their pair tables) on the device.  After set_trajectories every core
// is uploaded; after per-chunk updates only the changed ones travel: the new version is a device-to-device copy of the
// current one plus an expand of the updated records (parameters cross the bus only when they change).
// Work just enqueued on `stream` reads table version v.
static cudaError_t note_use(awg_plan *p, int v, cudaStream_t stream)
{
    awg_plan::VersionUse &u = p->use[v];
    cudaError_t e;
    int i = 0;
    while (i < u.n && u.stream[i] != stream) ++i;
    if (i == u.n) {
        if (u.n < kUseSlots) {
            if (!u.ev[i] && (e = cudaEventCreateWithFlags(&u.ev[i], cudaEventDisableTiming)) != cudaSuccess) return e;
            u.n++;
        } else {
            i = 0;   // more streams than slots: slot 0 changes hands once its own stream's work on this version is done
            if ((e = cudaEventSynchronize(u.ev[0])) != cudaSuccess) return e;
        }
        u.stream[i] = stream;
    }
    return cudaEventRecord(u.ev[i], stream);
}

// Blocks until every launch that reads table version v has finished (the version is about to be rewritten or freed).
static cudaError_t wait_users(awg_plan *p, int v)
{
    awg_plan::VersionUse &u = p->use[v];
    for (int i = 0; i < u.n; ++i) {
        cudaError_t e = cudaEventSynchronize(u.ev[i]);
        if (e != cudaSuccess) return e;
    }
    u.n = 0;
    return cudaSuccess;
}

awg_status ensure_table(awg_plan *p, cudaStream_t stream)
{
    cudaError_t e;
    if (!p->dirty_all && p->dirty_tones.empty()) {
        if (p->upload_stream[p->cur_version] != stream &&
            (e = cudaStreamWaitEvent(stream, p->uploaded[p->cur_version], 0)) != cudaSuccess)
            return fail_cuda(e, "cudaStreamWaitEvent");
        return AWG_OK;
    }
    const int cur = p->cur_version;
    const int v = (cur + 1) % kTableVersions;
    // the slot's previous readers (kernels launched kTableVersions uploads ago) must be done
    if ((e = wait_users(p, v)) != cudaSuccess) return fail_cuda(e, "cudaEventSynchronize");
    {
        std::vector<float> amp;
        amp.reserve(p->n_tones);
        for (int k = 0; k < p->n_tones; ++k)
            if (!p->in_buffer[k]) amp.push_back(std::max(std::fabs(p->tones[k].A), std::fabs(p->tones[k].A1)));
        fix_grids(amp.data(), static_cast<int>(amp.size()), &p->fix);
        p->slow2 = false;
        for (int k = 0; k < p->n_tones; ++k)
            if (!p->in_buffer[k] && (p->tones[k].cls & CLS_SLOW2_FLAG)) p->slow2 = true;
        p->hot_dirty = true;
    }
    std::sort(p->dirty_tones.begin(), p->dirty_tones.end());
    p->dirty_tones.erase(std::unique(p->dirty_tones.begin(), p->dirty_tones.end()), p->dirty_tones.end());
    const size_t n_dirty = p->dirty_tones.size();
    ToneCore *host = reinterpret_cast<ToneCore *>(p->host_table[v]);
    ToneRec *table = reinterpret_cast<ToneRec *>(p->dev_table[v]);
    const ToneCore *stage = reinterpret_cast<const ToneCore *>(p->dev_stage[v]);
    if (p->dirty_all || n_dirty * 2 > static_cast<size_t>(p->n_tones)) {
        // the device table holds the tones that are evaluated per sample (all of them unless some are served by the
        // looped static buffer), in tone order
        int n_act = 0;
        for (int k = 0; k < p->n_tones; ++k) p->slot_of[k] = p->in_buffer[k] ? -1 : n_act++;
        if (p->n_tones < kThreadedFrom) {
            for (int k = 0; k < p->n_tones; ++k)
                if (p->slot_of[k] >= 0) fill_core(p->tones[k], host[p->slot_of[k]]);
        } else {
            parallel_tones(p->n_tones, 1024, [=](int k_begin, int k_end) {
                for (int k = k_begin; k < k_end; ++k)
                    if (p->slot_of[k] >= 0) fill_core(p->tones[k], host[p->slot_of[k]]);
            });
        }
        p->n_active = n_act;
        const int n_up = (n_act + 31) / 32 * 32;
        for (int i = n_act; i < n_up; ++i) std::memset(&host[i], 0, sizeof(ToneCore));
        if (n_up > 0) {
            if ((e = cudaMemcpyAsync(p->dev_stage[v], host, static_cast<size_t>(n_up) * sizeof(ToneCore), cudaMemcpyHostToDevice, stream)) != cudaSuccess)
                return fail_cuda(e, "cudaMemcpyAsync(tone cores)");
            if ((e = launch_expand(table, stage, nullptr, n_up, stream)) != cudaSuccess) return fail_cuda(e, "expand launch");
        }
        p->h2d_bytes += static_cast<int64_t>(n_up) * static_cast<int64_t>(sizeof(ToneCore));
    } else {
        int32_t *host_idx = reinterpret_cast<int32_t *>(p->host_table[v] + p->core_bytes);
        for (size_t j = 0; j < n_dirty; ++j) {
            fill_core(p->tones[p->dirty_tones[j]], host[j]);
            host_idx[j] = p->slot_of[p->dirty_tones[j]];   // updates of tones in the static buffer are rejected earlier
        }
        if (p->upload_stream[cur] != stream && (e = cudaStreamWaitEvent(stream, p->uploaded[cur], 0)) != cudaSuccess)
            return fail_cuda(e, "cudaStreamWaitEvent");
        if ((e = cudaMemcpyAsync(p->dev_table[v], p->dev_table[cur], p->table_bytes, cudaMemcpyDeviceToDevice, stream)) != cudaSuccess)
            return fail_cuda(e, "cudaMemcpyAsync(table d2d)");
        if ((e = note_use(p, cur, stream)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
        if ((e = cudaMemcpyAsync(p->dev_stage[v], host, n_dirty * sizeof(ToneCore), cudaMemcpyHostToDevice, stream)) != cudaSuccess ||
            (e = cudaMemcpyAsync(p->dev_stage[v] + p->core_bytes, host_idx, n_dirty * sizeof(int32_t), cudaMemcpyHostToDevice, stream)) != cudaSuccess)
            return fail_cuda(e, "cudaMemcpyAsync(updated tone cores)");
        if ((e = launch_expand(table, stage, reinterpret_cast<const int32_t *>(p->dev_stage[v] + p->core_bytes), static_cast<int>(n_dirty),
                               stream)) != cudaSuccess)
            return fail_cuda(e, "expand launch");
        p->h2d_bytes += static_cast<int64_t>(n_dirty * (sizeof(ToneCore) + sizeof(int32_t)));
    }
    if ((e = cudaEventRecord(p->uploaded[v], stream)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
    p->upload_stream[v] = stream;
    p->cur_version = v;
    p->dirty_all = false;
    p->dirty_tones.clear();
    return AWG_OK;
}

// Hot tiles of a launch (LaunchParams::hot): tiles of the range in which at least max(2, n/16) of the n evaluated tones
// enter or leave a SLOW move (CLS_SLOW_FLAG).  Inside the move such a tone costs 1.25 multiply-adds per sample; in the tile
// that holds the boundary it takes the one-sine-per-sample pass for the whole tile: when many do so at once (tweezer
// rearrangements move their tones in step; C3: 1000 moves end in one tile) the tile costs several ordinary ones, and drawn in
// its turn it ended 0.15 ms after every other CTA had run out of work (C3: 1.69 -> 1.57 ms with the tile served first).
// The boundaries are a property of the table: they are listed once per table change (p->hot_tiles, absolute tile indices
// with their tone counts) and filtered per launch.  Fast movers are left out: their tiles cost the same inside the move.
static void list_hot_tiles(awg_plan *p)
{
    p->hot_tiles.clear();
    p->hot_dirty = false;
    if (p->n_active > 16384) return;
    static_assert((kTile & (kTile - 1)) == 0, "tile index = sample index >> log2(kTile), also for negative indices");
    constexpr int kTileShift = 11;
    static_assert((1 << kTileShift) == kTile, "kTileShift");
    // move starts and move ends, each in tone order: tones that move in step give long runs of equal keys, already in order
    std::vector<int64_t> (&at)[2] = p->hot_scratch;
    bool sorted[2] = {true, true};
    at[0].clear();
    at[1].clear();
    for (int k = 0; k < p->n_tones; ++k) {
        const HostTone &h = p->tones[k];
        if (!(h.cls & CLS_SLOW_FLAG) || p->in_buffer[k]) continue;
        // slow moves last >= 2 tiles and |t_start| fs < 4e18 (checked on entry): everything fits int64
        const int64_t t[2] = {h.ns_int >> kTileShift,
                              (h.ns_int + static_cast<int64_t>(static_cast<long double>(h.ns_frac) + h.Tn)) >> kTileShift};
        for (int e = 0; e < 2; ++e) {
            if (!at[e].empty() && t[e] < at[e].back()) sorted[e] = false;
            at[e].push_back(t[e]);
        }
    }
    if (at[0].empty()) return;
    const size_t thr = std::max<size_t>(2, static_cast<size_t>(p->n_active) / 16);
    std::vector<std::pair<int64_t, int64_t>> &runs = p->hot_tiles;   // (tile, tones), starts and ends counted separately at first
    for (int e = 0; e < 2; ++e) {
        if (!sorted[e]) std::sort(at[e].begin(), at[e].end());
        for (size_t i = 0; i < at[e].size();) {
            size_t j = i;
            while (j < at[e].size() && at[e][j] == at[e][i]) ++j;
            runs.emplace_back(at[e][i], static_cast<int64_t>(j - i));
            i = j;
        }
    }
    // a tile can hold starts and ends: add them up, then keep the tiles at or above the threshold
    std::sort(runs.begin(), runs.end());
    size_t n_out = 0;
    for (size_t i = 0; i < runs.size();) {
        size_t j = i;
        int64_t cnt = 0;
        while (j < runs.size() && runs[j].first == runs[i].first) cnt += runs[j++].second;
        if (static_cast<size_t>(cnt) >= thr) runs[n_out++] = std::make_pair(runs[i].first, cnt);
        i = j;
    }
    runs.resize(n_out);
}

static void find_hot_tiles(awg_plan *p, int64_t n_begin, int64_t n_count, LaunchParams &lp)
{
    lp.n_hot = 0;
    const int64_t first = n_begin / kTile, last = (n_begin + n_count - 1) / kTile;
    if (last - first + 1 < 64) return;   // every unit of such a launch starts at once anyway
    if (p->hot_dirty) list_hot_tiles(p);
    if (p->hot_tiles.empty()) return;
    std::pair<int64_t, int64_t> in[kMaxHotTiles];   // (tones, tile relative to the launch): the kMaxHotTiles heaviest of the range
    int n = 0;
    for (const auto &ht : p->hot_tiles) {
        if (ht.first < first || ht.first > last) continue;
        const std::pair<int64_t, int64_t> cand(ht.second, ht.first - first);
        if (n < kMaxHotTiles) {
            in[n++] = cand;
        } else {
            int m = 0;
            for (int i = 1; i < n; ++i)
                if (in[i].first < in[m].first) m = i;
            if (cand.first > in[m].first) in[m] = cand;
        }
    }
    std::sort(in, in + n, [](const std::pair<int64_t, int64_t> &a, const std::pair<int64_t, int64_t> &b) { return a.second < b.second; });
    for (int i = 0; i < n; ++i) lp.hot[lp.n_hot++] = static_cast<int32_t>(in[i].second);
}

awg_status synthesize_samples(awg_plan *p, int64_t n_begin, int64_t n_count, void *dev_out, bool f32, cudaStream_t stream,
                              int32_t out_stride, int32_t out_offset)
{
    awg_status st = ensure_table(p, stream);
    if (st != AWG_OK) return st;
    LaunchParams lp;
    lp.tab = reinterpret_cast<const ToneRec *>(p->dev_table[p->cur_version]);
    lp.n_tones = p->n_active;
    lp.out_stride = out_stride;
    lp.out_offset = out_offset;
    lp.xs = p->xs_on ? p->xs[p->xs_cur] : nullptr;
    lp.xs_len = p->chunk_len;
    lp.n_begin = n_begin;
    lp.n_count = n_count;
    lp.scale = static_cast<float>(p->scale);
    lp.fix = p->fix;
    lp.slow2 = p->slow2 ? 1 : 0;
    lp.out = dev_out;
    lp.out_f32 = f32 ? 1 : 0;
    lp.sched = nullptr;  // launch_synth assigns the tile-scheduler slot
    find_hot_tiles(p, n_begin, n_count, lp);
    cudaError_t e = launch_synth(lp, p->engine, stream);
    if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
    if ((e = note_use(p, p->cur_version, stream)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
    return AWG_OK;
}

// A plan lives on the device that was current when it was created; calls that enqueue work must be made with that
// device current (the library never switches devices behind the caller's back).
awg_status check_device(const awg_plan *p)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
    if (dev != p->device)
        return fail(AWG_ERR_STATE, "the plan was created on device %d but device %d is current", p->device, dev);
    return AWG_OK;
}

awg_status check_chunk_call(awg_plan *p, int64_t first_chunk, int64_t n_chunks, const void *out, size_t align)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (!out) return fail(AWG_ERR_INVALID_ARG, "output pointer is NULL");
    awg_status dst = check_device(p);
    if (dst != AWG_OK) return dst;
    if (reinterpret_cast<uintptr_t>(out) % align) return fail(AWG_ERR_INVALID_ARG, "output pointer must be %zu-byte aligned", align);
    if (first_chunk < 0 || n_chunks < 1) return fail(AWG_ERR_INVALID_ARG, "bad chunk range");
    if (first_chunk > (std::numeric_limits<int64_t>::max() / 4) / p->chunk_len - n_chunks)
        return fail(AWG_ERR_INVALID_ARG, "chunk index too large");
    if (!p->have_table) return fail(AWG_ERR_STATE, "awg_set_trajectories has not been called");
    if (first_chunk < p->last_update_chunk)
        return fail(AWG_ERR_STATE, "chunk %lld precedes the latest trajectory update (chunk %lld)",
                    static_cast<long long>(first_chunk), static_cast<long long>(p->last_update_chunk));
    return AWG_OK;
}

// awg_update_trajectories at sample n_u for the updates [i_begin, i_end) of one call (validated by the caller; the tones of one
// update are distinct, so every iteration has its own tone)
static inline __attribute__((always_inline)) void update_tones(awg_plan *p, int64_t n_u, const int32_t *tone_idx, const double *f1, const double *t_dur,
                         const int32_t *profile, int i_begin, int i_end)
{
    const long double fs = p->fs;
    for (int i = i_begin; i < i_end; ++i) {
        HostTone &h = p->tones[tone_idx[i]];
        // an amplitude ramp that has ended by n_u is folded into the tone's amplitude (the tables then carry it)
        if (h.amp_prof != AWG_PROFILE_STATIC && static_cast<long double>(n_u) - h.amp_ns >= h.amp_Tn) {
            h.A = h.A1;
            h.amp_prof = AWG_PROFILE_STATIC;
        }
        // state of the old segment at n_u: instantaneous frequency and a carrier that continues its phase
        if ((h.cls & 0xff) != CLS_STATIC) {
            const long double u = static_cast<long double>(n_u - h.ns_int) - static_cast<long double>(h.ns_frac);
            if (u <= 0.0L) {
                // move had not started: keep the pre-move carrier
            } else if (u >= h.Tn) {
                h.theta_pre = h.theta_post;
                h.w_pre = h.w_post;
                h.f0 = h.f1;
            } else {
                // mid-move (G12): continue from the instantaneous frequency and phase
                const long double s = u / h.Tn;
                const bool ex = h.profile == AWG_PROFILE_EXP;
                const long double f_now = ex ? h.f0 * expl(h.expL * s) : h.f0 + (h.f1 - h.f0) * profile_h(h.profile, s);
                const long double gain = ex ? h.f0 * h.T * (expm1l(h.expL * s) / h.expL - s) : h.DT * profile_g(h.profile, s);
                const uint64_t ph = h.theta_pre + h.w_pre * static_cast<uint64_t>(n_u) + frac64(gain);
                h.f0 = f_now;
                h.w_pre = frac64(f_now / fs);
                h.theta_pre = ph - h.w_pre * static_cast<uint64_t>(n_u);
            }
        }
        const long double f1l = static_cast<long double>(f1[i]);
        const long double D = f1l - h.f0;
        // (f1-f0) * t_u with t_u = n_u/fs
        make_move(h, fs, f1l, profile[i], static_cast<long double>(t_dur[i]), n_u, 0.0,
                  D * static_cast<long double>(n_u) / fs);
    }
}

awg_status apply_update(awg_plan *p, int64_t chunk_idx, int32_t n_upd, const int32_t *tone_idx, const double *f1,
                        const double *t_dur, const int32_t *profile)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (n_upd < 0 || chunk_idx < 0) return fail(AWG_ERR_INVALID_ARG, "negative count or chunk index");
    if (n_upd > 0 && (!tone_idx || !f1 || !t_dur || !profile)) return fail(AWG_ERR_INVALID_ARG, "NULL update array");
    if (!p->have_table) return fail(AWG_ERR_STATE, "awg_set_trajectories has not been called");
    if (chunk_idx < p->last_update_chunk)
        return fail(AWG_ERR_STATE, "updates must come in non-decreasing chunk order");
    if (chunk_idx > (std::numeric_limits<int64_t>::max() / 4) / p->chunk_len)
        return fail(AWG_ERR_INVALID_ARG, "chunk index too large");
    // validate everything before touching the table
    std::vector<char> seen(p->n_tones, 0);
    for (int i = 0; i < n_upd; ++i) {
        const int k = tone_idx[i];
        if (k < 0 || k >= p->n_tones) return fail(AWG_ERR_INVALID_ARG, "tone index %d out of range", k);
        if (seen[k]) return fail(AWG_ERR_INVALID_ARG, "tone %d listed twice in one update", k);
        seen[k] = 1;
        if (p->in_buffer[k]) return fail(AWG_ERR_STATE, "tone %d is served by the static buffer (clear it with awg_static_buffer_set first)", k);
        if (!std::isfinite(f1[i]) || !std::isfinite(t_dur[i]) || t_dur[i] < 0.0)
            return fail(AWG_ERR_INVALID_ARG, "non-finite value or negative duration in update %d", i);
        if (profile[i] < AWG_PROFILE_STATIC || profile[i] > AWG_PROFILE_EXP)
            return fail(AWG_ERR_INVALID_ARG, "unknown profile %d", profile[i]);
        if (profile[i] == AWG_PROFILE_EXP && !(f1[i] > 0.0 && p->tones[k].f0 > 0.0L && p->tones[k].f1 > 0.0L))
            return fail(AWG_ERR_INVALID_ARG, "exponential chirp of tone %d needs positive frequencies", k);
    }
    const int64_t n_u = chunk_idx * p->chunk_len;
    if (n_upd < kThreadedFrom) update_tones(p, n_u, tone_idx, f1, t_dur, profile, 0, n_upd);
    else parallel_tones(n_upd, 512, [=](int i_begin, int i_end) { update_tones(p, n_u, tone_idx, f1, t_dur, profile, i_begin, i_end); });
    if (n_upd > 0) {
        p->dirty_tones.insert(p->dirty_tones.end(), tone_idx, tone_idx + n_upd);
        p->last_update_chunk = chunk_idx;
    }
    return AWG_OK;
}

}  // namespace awg

using namespace awg;

extern "C" {

const char *awg_last_error(void) { return g_err; }

awg_status awg_plan_create(awg_plan **out, int32_t n_tones, double sample_rate_hz, int64_t chunk_len)
{
    if (!out) return fail(AWG_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (n_tones < 1 || n_tones > 65536) return fail(AWG_ERR_INVALID_ARG, "n_tones must be in [1, 65536]");
    if (!std::isfinite(sample_rate_hz) || sample_rate_hz <= 0.0) return fail(AWG_ERR_INVALID_ARG, "sample_rate_hz must be finite and > 0");
    if (chunk_len < 8 || chunk_len % 8 || chunk_len > (int64_t(1) << 40)) return fail(AWG_ERR_INVALID_ARG, "chunk_len must be a positive multiple of 8");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
    awg_plan *p = new (std::nothrow) awg_plan();
    if (!p) return fail(AWG_ERR_ALLOC, "out of host memory");
    p->n_tones = n_tones;
    p->n_pad = (n_tones + 31) / 32 * 32;
    p->fs = static_cast<long double>(sample_rate_hz);
    p->chunk_len = chunk_len;
    p->scale = 0.9 * 32767.0;
    p->engine = AWG_ENGINE_FMA;
    p->device = dev;
    p->table_bytes = static_cast<size_t>(p->n_pad) * sizeof(ToneRec);
    p->core_bytes = static_cast<size_t>(p->n_pad) * sizeof(ToneCore);
    try {
        p->tones.resize(n_tones);
        p->in_buffer.assign(n_tones, 0);
        p->slot_of.assign(n_tones, -1);
    } catch (...) {
        delete p;
        return fail(AWG_ERR_ALLOC, "out of host memory");
    }
    for (int v = 0; v < kTableVersions; ++v) {
        const size_t stage_bytes = p->core_bytes + static_cast<size_t>(p->n_pad) * sizeof(int32_t);
        if ((e = cudaMalloc(reinterpret_cast<void **>(&p->dev_table[v]), p->table_bytes)) != cudaSuccess ||
            (e = cudaMalloc(reinterpret_cast<void **>(&p->dev_stage[v]), stage_bytes)) != cudaSuccess ||
            (e = cudaMallocHost(reinterpret_cast<void **>(&p->host_table[v]), stage_bytes)) != cudaSuccess ||
            (e = cudaEventCreateWithFlags(&p->uploaded[v], cudaEventDisableTiming)) != cudaSuccess) {
            awg_status st = (e == cudaErrorMemoryAllocation) ? fail(AWG_ERR_ALLOC, "device/pinned allocation failed: %s", cudaGetErrorString(e))
                                                             : fail_cuda(e, "plan allocation");
            awg_plan_destroy(p);
            return st;
        }
    }
    *out = p;
    return AWG_OK;
}

static void free_e2e(awg_plan *p)
{
    for (int s = 0; s < kE2eSlots; ++s) {
        if (p->e2e_slot[s]) cudaFree(p->e2e_slot[s]);
        if (p->e2e_done[s]) cudaEventDestroy(p->e2e_done[s]);
        if (p->e2e_ready[s]) cudaEventDestroy(p->e2e_ready[s]);
        p->e2e_slot[s] = nullptr; p->e2e_done[s] = nullptr; p->e2e_ready[s] = nullptr;
    }
    for (int s = 0; s < 3; ++s) {
        if (p->e2e_stream[s]) cudaStreamDestroy(p->e2e_stream[s]);
        p->e2e_stream[s] = nullptr;
    }
}

awg_status awg_plan_destroy(awg_plan *p)
{
    if (!p) return AWG_OK;
    if (p->n_rings > 0) return fail(AWG_ERR_STATE, "destroy the plan's rings first");
    for (int v = 0; v < kTableVersions; ++v)
        (void)wait_users(p, v);
    for (int s = 0; s < kE2eSlots; ++s) {
        if (p->e2e_done[s]) cudaEventSynchronize(p->e2e_done[s]);
    }
    for (int v = 0; v < kTableVersions; ++v) {
        if (p->dev_table[v]) cudaFree(p->dev_table[v]);
        if (p->dev_stage[v]) cudaFree(p->dev_stage[v]);
        if (p->host_table[v]) cudaFreeHost(p->host_table[v]);
        for (int i = 0; i < kUseSlots; ++i)
            if (p->use[v].ev[i]) cudaEventDestroy(p->use[v].ev[i]);
        if (p->uploaded[v]) cudaEventDestroy(p->uploaded[v]);
    }
    for (int s = 0; s < 2; ++s)
        if (p->xs[s]) cudaFree(p->xs[s]);
    if (p->dev_aux) cudaFree(p->dev_aux);
    if (p->dev_aux_stage) cudaFree(p->dev_aux_stage);
    if (p->host_aux) cudaFreeHost(p->host_aux);
    free_e2e(p);
    for (int i = 0; i < p->mux_n; ++i) {
        cudaStreamSynchronize(p->mux_stream[i]);
        cudaStreamDestroy(p->mux_stream[i]);
        cudaEventDestroy(p->mux_join[i]);
    }
    if (p->mux_fork) cudaEventDestroy(p->mux_fork);
    delete p;
    return AWG_OK;
}

awg_status awg_plan_io_bytes(awg_plan *p, int64_t *h2d_bytes, int64_t *d2h_bytes)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (h2d_bytes) *h2d_bytes = p->h2d_bytes;
    if (d2h_bytes) *d2h_bytes = p->d2h_bytes;
    return AWG_OK;
}

awg_status awg_plan_hot_tiles(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int32_t *n_listed, int32_t *n_served_first)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (first_chunk < 0 || n_chunks < 1) return fail(AWG_ERR_INVALID_ARG, "bad chunk range");
    if (!p->have_table) return fail(AWG_ERR_STATE, "awg_set_trajectories has not been called");
    list_hot_tiles(p);   // from the host table as it stands (per-chunk updates included)
    const int64_t n0 = first_chunk * p->chunk_len, cnt = n_chunks * p->chunk_len;
    const int64_t first = n0 / kTile, last = (n0 + cnt - 1) / kTile;
    int32_t listed = 0;
    for (const auto &ht : p->hot_tiles)
        if (ht.first >= first && ht.first <= last) ++listed;
    LaunchParams lp;
    find_hot_tiles(p, n0, cnt, lp);
    if (n_listed) *n_listed = listed;
    if (n_served_first) *n_served_first = lp.n_hot;
    return AWG_OK;
}

awg_status awg_plan_op_counts(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int64_t *static_ts, int64_t *slow_ts, int64_t *fast_ts)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (first_chunk < 0 || n_chunks < 0) return fail(AWG_ERR_INVALID_ARG, "bad chunk range");
    if (!p->have_table) return fail(AWG_ERR_STATE, "awg_set_trajectories has not been called");
    const int64_t n0 = first_chunk * p->chunk_len, n1 = n0 + n_chunks * p->chunk_len;
    int64_t n_static = 0, n_slow = 0, n_fast = 0;
    for (int k = 0; k < p->n_tones; ++k) {
        if (p->in_buffer[k]) continue;   // served by the looped static buffer: no per-sample work
        const HostTone &h = p->tones[k];
        int64_t moving = 0;
        if ((h.cls & 0xff) != CLS_STATIC) {
            // samples n with 0 < u < Tn, u = (n - ns_int) - ns_frac
            const long double ns = static_cast<long double>(h.ns_int) + static_cast<long double>(h.ns_frac);
            const int64_t first = static_cast<int64_t>(floorl(ns)) + 1;
            const int64_t last = static_cast<int64_t>(ceill(ns + h.Tn)) - 1;
            const int64_t a = first > n0 ? first : n0, b = last < n1 - 1 ? last : n1 - 1;
            if (b >= a) moving = b - a + 1;
        }
        int64_t ramping = 0;   // samples inside an amplitude ramp are evaluated one by one as well
        if (h.amp_prof != AWG_PROFILE_STATIC) {
            const int64_t first = static_cast<int64_t>(floorl(h.amp_ns)) + 1;
            const int64_t last = static_cast<int64_t>(ceill(h.amp_ns + h.amp_Tn)) - 1;
            const int64_t a = first > n0 ? first : n0, b = last < n1 - 1 ? last : n1 - 1;
            if (b >= a) ramping = b - a + 1;
        }
        if (ramping > 0) {
            // (the union of the two windows is what leaves the angle-addition engine; counted as the larger one)
            if (ramping > moving) { n_fast += ramping; moving = ramping; }
            else if (h.cls & CLS_SLOW_FLAG) n_fast += moving;
            else n_fast += moving;
        } else if (h.cls & CLS_SLOW_FLAG) {
            n_slow += moving;
        } else {
            n_fast += moving;
        }
        n_static += (n1 - n0) - moving;
    }
    if (static_ts) *static_ts = n_static;
    if (slow_ts) *slow_ts = n_slow;
    if (fast_ts) *fast_ts = n_fast;
    return AWG_OK;
}

// ---- static-buffer pathway (section IV A/B of the paper) ------------------------------------------------------

awg_status awg_snap_frequency(double f0_hz, double sample_rate_hz, int64_t L_s, double *f_snapped_hz)
{
    if (!f_snapped_hz) return fail(AWG_ERR_INVALID_ARG, "f_snapped_hz is NULL");
    if (!std::isfinite(f0_hz) || !std::isfinite(sample_rate_hz) || sample_rate_hz <= 0.0 || L_s < 1)
        return fail(AWG_ERR_INVALID_ARG, "bad frequency, rate or buffer length");
    // Eq. 6: f_j = nint(f0 L_s / fs) fs / L_s
    const long double fs = sample_rate_hz, L = static_cast<long double>(L_s);
    *f_snapped_hz = static_cast<double>(rintl(static_cast<long double>(f0_hz) * L / fs) * fs / L);
    return AWG_OK;
}

namespace awg {
namespace {

// does the carrier frequency w (turns * 2^64 per sample) make a whole number of turns in L samples?  (Eq. 5/6)  The
// frequency arrived as a double: its rounding (2^-53 relative, f/fs < 1) is allowed for, i.e. a phase drift of at most
// L 2^-53 turns per period, far below anything the output resolves.
bool periodic_in(uint64_t w, int64_t L)
{
    const int64_t r = static_cast<int64_t>(w * static_cast<uint64_t>(L));
    return r <= 2048 * L && r >= -2048 * L;
}

awg_status static_buffer_alloc(awg_plan *p)
{
    cudaError_t e;
    const size_t bytes = static_cast<size_t>(p->chunk_len) * sizeof(float);
    for (int s = 0; s < 2; ++s)
        if (!p->xs[s] && (e = cudaMalloc(reinterpret_cast<void **>(&p->xs[s]), bytes)) != cudaSuccess)
            return fail(AWG_ERR_ALLOC, "cudaMalloc(static buffer): %s", cudaGetErrorString(e));
    const size_t stage_bytes = p->core_bytes + static_cast<size_t>(p->n_pad) * sizeof(int32_t);
    if (!p->dev_aux && (e = cudaMalloc(reinterpret_cast<void **>(&p->dev_aux), p->table_bytes)) != cudaSuccess)
        return fail(AWG_ERR_ALLOC, "cudaMalloc(static-buffer table): %s", cudaGetErrorString(e));
    if (!p->dev_aux_stage && (e = cudaMalloc(reinterpret_cast<void **>(&p->dev_aux_stage), stage_bytes)) != cudaSuccess)
        return fail(AWG_ERR_ALLOC, "cudaMalloc(static-buffer staging): %s", cudaGetErrorString(e));
    if (!p->host_aux && (e = cudaMallocHost(reinterpret_cast<void **>(&p->host_aux), stage_bytes)) != cudaSuccess)
        return fail(AWG_ERR_ALLOC, "cudaMallocHost(static-buffer staging): %s", cudaGetErrorString(e));
    return AWG_OK;
}

// One period [0, L_s) of the static carriers `tones` is synthesised as fp32 (the synthesis kernel, fp32 output) into
// `dst`, on top of `base` when that is not NULL (Eq. 8; Eq. 10 branch 3).  Synchronous.
awg_status static_buffer_add(awg_plan *p, const std::vector<HostTone> &tones, const float *base, float *dst, cudaStream_t stream)
{
    cudaError_t e;
    const int n = static_cast<int>(tones.size());
    const int n_up = (n + 31) / 32 * 32;
    ToneCore *host = reinterpret_cast<ToneCore *>(p->host_aux);
    for (int i = 0; i < n_up; ++i) {
        if (i < n) fill_core(tones[i], host[i]);
        else std::memset(&host[i], 0, sizeof(ToneCore));
    }
    if ((e = cudaMemcpyAsync(p->dev_aux_stage, host, static_cast<size_t>(n_up) * sizeof(ToneCore), cudaMemcpyHostToDevice, stream)) != cudaSuccess)
        return fail_cuda(e, "cudaMemcpyAsync(static-buffer cores)");
    if ((e = launch_expand(reinterpret_cast<ToneRec *>(p->dev_aux), reinterpret_cast<const ToneCore *>(p->dev_aux_stage), nullptr, n_up,
                           stream)) != cudaSuccess)
        return fail_cuda(e, "expand launch");
    p->h2d_bytes += static_cast<int64_t>(n_up) * static_cast<int64_t>(sizeof(ToneCore));
    LaunchParams lp;
    lp.tab = reinterpret_cast<const ToneRec *>(p->dev_aux);
    lp.n_tones = n;
    lp.out_f32 = 1;
    lp.n_begin = 0;
    lp.n_count = p->chunk_len;
    lp.scale = static_cast<float>(p->scale);
    std::vector<float> amp;
    for (const HostTone &h : tones) amp.push_back(std::max(std::fabs(h.A), std::fabs(h.A1)));
    fix_grids(amp.data(), n, &lp.fix);
    lp.slow2 = 0;   // (static carriers only)
    lp.out = dst;
    lp.out_stride = 1;
    lp.out_offset = 0;
    lp.xs = base;
    lp.xs_len = p->chunk_len;
    lp.sched = nullptr;
    if ((e = launch_synth(lp, p->engine, stream)) != cudaSuccess) return fail_cuda(e, "kernel launch");
    if ((e = cudaStreamSynchronize(stream)) != cudaSuccess) return fail_cuda(e, "cudaStreamSynchronize");
    return AWG_OK;
}

awg_status check_tone_list(awg_plan *p, int32_t n, const int32_t *tone_idx)
{
    if (n < 0 || (n > 0 && !tone_idx)) return fail(AWG_ERR_INVALID_ARG, "bad tone list");
    std::vector<char> seen(p->n_tones, 0);
    for (int i = 0; i < n; ++i) {
        const int k = tone_idx[i];
        if (k < 0 || k >= p->n_tones) return fail(AWG_ERR_INVALID_ARG, "tone index %d out of range", k);
        if (seen[k]) return fail(AWG_ERR_INVALID_ARG, "tone %d listed twice", k);
        seen[k] = 1;
    }
    return AWG_OK;
}

}  // namespace
}  // namespace awg

awg_status awg_static_buffer_set(awg_plan *p, int32_t n_static, const int32_t *tone_idx, void *stream)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    awg_status st = check_device(p);
    if (st != AWG_OK) return st;
    if (!p->have_table) return fail(AWG_ERR_STATE, "awg_set_trajectories has not been called");
    if ((st = check_tone_list(p, n_static, tone_idx)) != AWG_OK) return st;
    if (n_static == 0) {   // back to evaluating every tone per sample
        std::fill(p->in_buffer.begin(), p->in_buffer.end(), 0);
        p->xs_on = false;
        p->dirty_all = true;
        return AWG_OK;
    }
    if (p->chunk_len < kTile) return fail(AWG_ERR_INVALID_ARG, "the static-buffer pathway needs chunk_len >= %d", kTile);
    std::vector<HostTone> tones;
    for (int i = 0; i < n_static; ++i) {
        const HostTone &h = p->tones[tone_idx[i]];
        if ((h.cls & 0xff) != CLS_STATIC || h.amp_prof != AWG_PROFILE_STATIC)
            return fail(AWG_ERR_INVALID_ARG, "tone %d is not static", tone_idx[i]);
        if (!periodic_in(h.w_pre, p->chunk_len))
            return fail(AWG_ERR_INVALID_ARG, "tone %d is off the fs/L_s grid (Eq. 6): snap it with awg_snap_frequency", tone_idx[i]);
        tones.push_back(h);
    }
    if ((st = static_buffer_alloc(p)) != AWG_OK) return st;
    if ((st = static_buffer_add(p, tones, nullptr, p->xs[0], static_cast<cudaStream_t>(stream))) != AWG_OK) return st;
    std::fill(p->in_buffer.begin(), p->in_buffer.end(), 0);
    for (int i = 0; i < n_static; ++i) p->in_buffer[tone_idx[i]] = 1;
    p->xs_cur = 0;
    p->xs_on = true;
    p->dirty_all = true;
    return AWG_OK;
}

awg_status awg_static_buffer_fold(awg_plan *p, int64_t chunk_idx, int32_t n_fold, const int32_t *tone_idx, void *stream)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    awg_status st = check_device(p);
    if (st != AWG_OK) return st;
    if (!p->have_table) return fail(AWG_ERR_STATE, "awg_set_trajectories has not been called");
    if (chunk_idx < 0 || chunk_idx > (std::numeric_limits<int64_t>::max() / 4) / p->chunk_len)
        return fail(AWG_ERR_INVALID_ARG, "bad chunk index");
    if (chunk_idx < p->last_update_chunk) return fail(AWG_ERR_STATE, "the hand-back precedes the latest trajectory update");
    if ((st = check_tone_list(p, n_fold, tone_idx)) != AWG_OK) return st;
    if (n_fold == 0) return AWG_OK;
    if (p->chunk_len < kTile) return fail(AWG_ERR_INVALID_ARG, "the static-buffer pathway needs chunk_len >= %d", kTile);
    const int64_t n_d = chunk_idx * p->chunk_len;   // L_d: a multiple of L_s
    std::vector<HostTone> tones;
    for (int i = 0; i < n_fold; ++i) {
        const int k = tone_idx[i];
        if (p->in_buffer[k]) return fail(AWG_ERR_STATE, "tone %d is already in the static buffer", k);
        HostTone h = p->tones[k];
        if (h.amp_prof != AWG_PROFILE_STATIC) {
            const long double ua = static_cast<long double>(n_d) - h.amp_ns;
            if (ua > 0.0L && ua < h.amp_Tn)
                return fail(AWG_ERR_STATE, "tone %d is inside its amplitude ramp at the hand-back (chunk %lld)", k, static_cast<long long>(chunk_idx));
            if (ua >= h.amp_Tn) h.A = h.A1;
            h.A1 = h.A;
            h.amp_prof = AWG_PROFILE_STATIC;
        }
        if ((h.cls & 0xff) != CLS_STATIC) {
            const long double u = static_cast<long double>(n_d - h.ns_int) - static_cast<long double>(h.ns_frac);
            if (u <= 0.0L) {
                // the move has not begun: the tone is still on its first carrier
            } else if (u >= h.Tn) {
                h.theta_pre = h.theta_post;   // theta' of Eq. 10 is this carrier's phase at L_d
                h.w_pre = h.w_post;
                h.f0 = h.f1;
            } else {
                return fail(AWG_ERR_STATE, "tone %d is still moving at the hand-back (chunk %lld)", k, static_cast<long long>(chunk_idx));
            }
            make_static(h);
        }
        if (!periodic_in(h.w_pre, p->chunk_len))
            return fail(AWG_ERR_INVALID_ARG, "tone %d ends off the fs/L_s grid (Eq. 6): its looped wavetable would not be seamless", k);
        tones.push_back(h);
    }
    if ((st = static_buffer_alloc(p)) != AWG_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    if (!p->xs_on) {
        if ((e = cudaMemsetAsync(p->xs[0], 0, static_cast<size_t>(p->chunk_len) * sizeof(float), s)) != cudaSuccess)
            return fail_cuda(e, "cudaMemsetAsync");
        p->xs_cur = 0;
    }
    // work in flight may still read the current buffer: the sum goes to the other one
    if ((st = static_buffer_add(p, tones, p->xs[p->xs_cur], p->xs[p->xs_cur ^ 1], s)) != AWG_OK) return st;
    p->xs_cur ^= 1;
    p->xs_on = true;
    for (int i = 0; i < n_fold; ++i) p->in_buffer[tone_idx[i]] = 1;
    p->dirty_all = true;
    p->last_update_chunk = chunk_idx;
    return AWG_OK;
}

awg_status awg_static_buffer_read(awg_plan *p, float *dev_out, void *stream)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (!dev_out) return fail(AWG_ERR_INVALID_ARG, "output pointer is NULL");
    awg_status st = check_device(p);
    if (st != AWG_OK) return st;
    if (!p->xs_on) return fail(AWG_ERR_STATE, "the plan has no static buffer");
    cudaError_t e = cudaMemcpyAsync(dev_out, p->xs[p->xs_cur], static_cast<size_t>(p->chunk_len) * sizeof(float), cudaMemcpyDeviceToDevice,
                                    static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "cudaMemcpyAsync");
    return AWG_OK;
}

// ---- four-channel multiplexed output (the paper's WM kernel) ------------------------------------------------------

awg_status awg_synthesize_chunk_mux(awg_plan *const *plans, int32_t n_channels, int64_t chunk_idx, int16_t *dev_out, void *stream)
{
    if (!plans) return fail(AWG_ERR_INVALID_ARG, "plans is NULL");
    if (n_channels < 1 || n_channels > 8) return fail(AWG_ERR_INVALID_ARG, "n_channels must be in [1, 8]");
    for (int c = 0; c < n_channels; ++c) {
        if (!plans[c]) return fail(AWG_ERR_INVALID_ARG, "plan of channel %d is NULL", c);
        if (plans[c]->chunk_len != plans[0]->chunk_len) return fail(AWG_ERR_INVALID_ARG, "the channels' plans must share chunk_len");
        for (int d = 0; d < c; ++d)
            if (plans[d] == plans[c]) return fail(AWG_ERR_INVALID_ARG, "channels %d and %d share a plan", d, c);
    }
    // validate every channel before the first launch
    for (int c = 0; c < n_channels; ++c) {
        awg_status st = check_chunk_call(plans[c], chunk_idx, 1, dev_out, 16);
        if (st != AWG_OK) return st;
    }
    // Channel 0 runs on the caller's stream, the others beside it on streams of their own (forked from and joined back into
    // the caller's stream with events): a channel of a few dozen tones is a launch of a few microseconds that uses a fraction
    // of the SMs, and four of them back to back on one stream take four times as long as side by side.
    awg_plan *p0 = plans[0];
    cudaStream_t user = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    if (n_channels > 1) {
        if (!p0->mux_fork && (e = cudaEventCreateWithFlags(&p0->mux_fork, cudaEventDisableTiming)) != cudaSuccess)
            return fail_cuda(e, "cudaEventCreate(mux)");
        while (p0->mux_n < n_channels - 1) {
            const int i = p0->mux_n;
            if ((e = cudaStreamCreateWithFlags(&p0->mux_stream[i], cudaStreamNonBlocking)) != cudaSuccess) return fail_cuda(e, "cudaStreamCreate(mux)");
            if ((e = cudaEventCreateWithFlags(&p0->mux_join[i], cudaEventDisableTiming)) != cudaSuccess) {
                cudaStreamDestroy(p0->mux_stream[i]);
                p0->mux_stream[i] = nullptr;
                return fail_cuda(e, "cudaEventCreate(mux)");
            }
            p0->mux_n = i + 1;
        }
        if ((e = cudaEventRecord(p0->mux_fork, user)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
    }
    awg_status first_bad = AWG_OK;
    int n_forked = 0;
    for (int c = 0; c < n_channels; ++c) {
        awg_plan *p = plans[c];
        cudaStream_t s = c == 0 ? user : p0->mux_stream[c - 1];
        if (c > 0 && (e = cudaStreamWaitEvent(s, p0->mux_fork, 0)) != cudaSuccess) {
            first_bad = fail_cuda(e, "cudaStreamWaitEvent");
            break;
        }
        awg_status st = synthesize_samples(p, chunk_idx * p->chunk_len, p->chunk_len, dev_out, false, s, n_channels, c);
        if (c > 0) n_forked = c;   // whatever was enqueued on the side stream is joined below, also after an error
        if (st != AWG_OK) {
            first_bad = st;
            break;
        }
    }
    for (int c = 1; c <= n_forked; ++c) {
        if ((e = cudaEventRecord(p0->mux_join[c - 1], p0->mux_stream[c - 1])) != cudaSuccess ||
            (e = cudaStreamWaitEvent(user, p0->mux_join[c - 1], 0)) != cudaSuccess)
            return fail_cuda(e, "mux join");
    }
    return first_bad;
}

awg_status awg_set_scale(awg_plan *p, double scale)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (!std::isfinite(scale) || scale <= 0.0) return fail(AWG_ERR_INVALID_ARG, "scale must be finite and > 0");
    p->scale = scale;
    return AWG_OK;
}

awg_status awg_set_engine(awg_plan *p, int32_t engine)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (engine == AWG_ENGINE_AUTO) engine = AWG_ENGINE_FMA;
    if (engine != AWG_ENGINE_MUFU && engine != AWG_ENGINE_FP64 && engine != AWG_ENGINE_FMA)
        return fail(AWG_ERR_INVALID_ARG, "unknown engine %d", engine);
    p->engine = engine;
    return AWG_OK;
}

// awg_set_trajectories for the tones [k_begin, k_end) (validated by the caller)
static inline __attribute__((always_inline)) void plan_tones(awg_plan *p, const double *f0, const double *f1, const double *A, const double *phi0, const double *t_start,
                       const double *t_dur, const int32_t *profile, int k_begin, int k_end)
{
    const long double fs = p->fs;
    for (int k = k_begin; k < k_end; ++k) {
        HostTone &h = p->tones[k];
        h = HostTone{};
        h.A = static_cast<float>(A[k]);
        h.A1 = h.A;
        h.f0 = static_cast<long double>(f0[k]);
        h.theta_pre = frac64(static_cast<long double>(phi0[k]) / kTwoPiL);  // radians -> turns (theta_j of Eq. 8/9)
        h.w_pre = frac64(h.f0 / fs);
        const long double ts = static_cast<long double>(t_start[k]);
        const long double ns = ts * fs;
        const long double nsi = floorl(ns);
        make_move(h, fs, static_cast<long double>(f1[k]), profile[k], static_cast<long double>(t_dur[k]),
                  static_cast<int64_t>(nsi), static_cast<double>(ns - nsi),
                  (static_cast<long double>(f1[k]) - h.f0) * ts);
    }
}

awg_status awg_set_trajectories(awg_plan *p, const double *f0, const double *f1, const double *A, const double *phi0,
                                const double *t_start, const double *t_dur, const int32_t *profile)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (!f0 || !f1 || !A || !phi0 || !t_start || !t_dur || !profile) return fail(AWG_ERR_INVALID_ARG, "NULL trajectory array");
    const int N = p->n_tones;
    if (!finite_all(f0, N) || !finite_all(f1, N) || !finite_all(A, N) || !finite_all(phi0, N) ||
        !finite_all(t_start, N) || !finite_all(t_dur, N))
        return fail(AWG_ERR_INVALID_ARG, "non-finite value in a trajectory array");
    for (int k = 0; k < N; ++k) {
        if (t_dur[k] < 0.0) return fail(AWG_ERR_INVALID_ARG, "t_dur[%d] < 0", k);
        if (profile[k] < AWG_PROFILE_STATIC || profile[k] > AWG_PROFILE_EXP)
            return fail(AWG_ERR_INVALID_ARG, "unknown profile %d for tone %d", profile[k], k);
        if (profile[k] == AWG_PROFILE_EXP && !(f0[k] > 0.0 && f1[k] > 0.0))
            return fail(AWG_ERR_INVALID_ARG, "exponential chirp of tone %d needs f0 > 0 and f1 > 0", k);
        if (std::fabs(t_start[k]) * static_cast<double>(p->fs) > 4.0e18)
            return fail(AWG_ERR_INVALID_ARG, "t_start[%d] out of range", k);
    }
    if (N < kThreadedFrom) plan_tones(p, f0, f1, A, phi0, t_start, t_dur, profile, 0, N);
    else parallel_tones(N, 512, [=](int k_begin, int k_end) { plan_tones(p, f0, f1, A, phi0, t_start, t_dur, profile, k_begin, k_end); });
    p->have_table = true;
    p->dirty_all = true;
    p->dirty_tones.clear();
    p->last_update_chunk = 0;
    std::fill(p->in_buffer.begin(), p->in_buffer.end(), 0);
    p->xs_on = false;
    return AWG_OK;
}

// ---- allocation-free one-shot synthesis (include/awg.h: awg_synthesize_noalloc) --------------------------------------
// No plan, hence no cudaMalloc: the host builds the tone cores into a static host array, and the table, the scheduler
// counters and the cross-CTA scratch tiles live in the library's static __device__ array (awg_kernels.cu).
static std::mutex g_noalloc_mutex;
static ToneCore g_noalloc_cores[kNoAllocMaxTones];   // host staging of the tone cores (0.5 MB of .bss)

awg_status awg_synthesize_noalloc(double sample_rate_hz, int32_t n_tones, const double *f0, const double *f1, const double *A,
                                  const double *phi0, const double *t_start, const double *t_dur, const int32_t *profile,
                                  int64_t first_sample, int64_t n_samples, int16_t *dev_out, void *stream)
{
    if (n_tones < 1 || n_tones > kNoAllocMaxTones)
        return fail(AWG_ERR_INVALID_ARG, "awg_synthesize_noalloc: n_tones = %d is outside [1, %d] (the static scratch holds %d tone records; use a plan for more)",
                    n_tones, kNoAllocMaxTones, kNoAllocMaxTones);
    if (n_samples < 8 || n_samples % 8 || n_samples > kNoAllocMaxSamples)
        return fail(AWG_ERR_INVALID_ARG, "awg_synthesize_noalloc: n_samples = %lld must be a multiple of 8 in [8, %lld] (the static scratch holds %lld samples per call; call again for the next range, or use a plan)",
                    static_cast<long long>(n_samples), static_cast<long long>(kNoAllocMaxSamples), static_cast<long long>(kNoAllocMaxSamples));
    if (first_sample < 0 || first_sample % 8 || first_sample > std::numeric_limits<int64_t>::max() / 4)
        return fail(AWG_ERR_INVALID_ARG, "awg_synthesize_noalloc: first_sample must be a multiple of 8 in [0, 2^61]");
    if (!std::isfinite(sample_rate_hz) || sample_rate_hz <= 0.0) return fail(AWG_ERR_INVALID_ARG, "sample_rate_hz must be finite and > 0");
    if (!f0 || !f1 || !A || !phi0 || !t_start || !t_dur || !profile) return fail(AWG_ERR_INVALID_ARG, "NULL trajectory array");
    if (!dev_out) return fail(AWG_ERR_INVALID_ARG, "output pointer is NULL");
    if (reinterpret_cast<uintptr_t>(dev_out) % 16) return fail(AWG_ERR_INVALID_ARG, "output pointer must be 16-byte aligned");
    const int N = n_tones;
    if (!finite_all(f0, N) || !finite_all(f1, N) || !finite_all(A, N) || !finite_all(phi0, N) || !finite_all(t_start, N) || !finite_all(t_dur, N))
        return fail(AWG_ERR_INVALID_ARG, "non-finite value in a trajectory array");
    for (int k = 0; k < N; ++k) {
        if (t_dur[k] < 0.0) return fail(AWG_ERR_INVALID_ARG, "t_dur[%d] < 0", k);
        if (profile[k] < AWG_PROFILE_STATIC || profile[k] > AWG_PROFILE_EXP) return fail(AWG_ERR_INVALID_ARG, "unknown profile %d for tone %d", profile[k], k);
        if (profile[k] == AWG_PROFILE_EXP && !(f0[k] > 0.0 && f1[k] > 0.0))
            return fail(AWG_ERR_INVALID_ARG, "exponential chirp of tone %d needs f0 > 0 and f1 > 0", k);
        if (std::fabs(t_start[k]) * sample_rate_hz > 4.0e18) return fail(AWG_ERR_INVALID_ARG, "t_start[%d] out of range", k);
    }
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);   // one host staging array
    const long double fs = static_cast<long double>(sample_rate_hz);
    float amp[kNoAllocMaxTones];
    bool slow2 = false;
    for (int k = 0; k < N; ++k) {
        // the tone of awg_set_trajectories, one at a time (no host table is kept)
        HostTone h{};
        h.A = static_cast<float>(A[k]);
        h.A1 = h.A;
        h.f0 = static_cast<long double>(f0[k]);
        h.theta_pre = frac64(static_cast<long double>(phi0[k]) / kTwoPiL);
        h.w_pre = frac64(h.f0 / fs);
        const long double ts = static_cast<long double>(t_start[k]);
        const long double ns = ts * fs;
        const long double nsi = floorl(ns);
        make_move(h, fs, static_cast<long double>(f1[k]), profile[k], static_cast<long double>(t_dur[k]), static_cast<int64_t>(nsi),
                  static_cast<double>(ns - nsi), (static_cast<long double>(f1[k]) - h.f0) * ts);
        fill_core(h, g_noalloc_cores[k]);
        amp[k] = std::fabs(h.A);
        if (h.cls & CLS_SLOW2_FLAG) slow2 = true;
    }
    const int n_up = (N + 31) / 32 * 32;
    for (int k = N; k < n_up; ++k) std::memset(&g_noalloc_cores[k], 0, sizeof(ToneCore));
    LaunchParams lp;
    lp.tab = nullptr;   // (launch_synth_noalloc: the table is built in the static device array)
    lp.n_tones = N;
    lp.out_stride = 1;
    lp.out_offset = 0;
    lp.xs = nullptr;
    lp.xs_len = 0;
    lp.n_begin = first_sample;
    lp.n_count = n_samples;
    lp.scale = static_cast<float>(0.9 * 32767.0);   // the default scale of a plan
    fix_grids(amp, N, &lp.fix);
    lp.slow2 = slow2 ? 1 : 0;
    lp.out = dev_out;
    lp.out_f32 = 0;
    lp.sched = nullptr;
    lp.n_hot = 0;
    const cudaError_t e = launch_synth_noalloc(g_noalloc_cores, n_up, lp, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "awg_synthesize_noalloc");
    return AWG_OK;
}

awg_status awg_set_amplitude_ramps(awg_plan *p, const double *A1, const double *t_start, const double *t_dur, const int32_t *profile)
{
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (!A1 || !t_start || !t_dur || !profile) return fail(AWG_ERR_INVALID_ARG, "NULL ramp array");
    if (!p->have_table) return fail(AWG_ERR_STATE, "awg_set_trajectories has not been called");
    if (p->last_update_chunk > 0) return fail(AWG_ERR_STATE, "amplitude ramps are set before the first trajectory update");
    const int N = p->n_tones;
    if (!finite_all(A1, N) || !finite_all(t_start, N) || !finite_all(t_dur, N)) return fail(AWG_ERR_INVALID_ARG, "non-finite value in a ramp array");
    for (int k = 0; k < N; ++k) {
        if (t_dur[k] < 0.0) return fail(AWG_ERR_INVALID_ARG, "t_dur[%d] < 0", k);
        if (profile[k] < AWG_PROFILE_STATIC || profile[k] > AWG_PROFILE_MINJERK)
            return fail(AWG_ERR_INVALID_ARG, "unknown profile %d for tone %d", profile[k], k);
        if (std::fabs(t_start[k]) * static_cast<double>(p->fs) > 4.0e18) return fail(AWG_ERR_INVALID_ARG, "t_start[%d] out of range", k);
        if (profile[k] != AWG_PROFILE_STATIC && p->in_buffer[k])
            return fail(AWG_ERR_STATE, "tone %d is served by the static buffer", k);
    }
    for (int k = 0; k < N; ++k) {
        HostTone &h = p->tones[k];
        h.amp_prof = profile[k];
        h.A1 = profile[k] == AWG_PROFILE_STATIC ? h.A : static_cast<float>(A1[k]);
        h.amp_ns = static_cast<long double>(t_start[k]) * p->fs;
        h.amp_Tn = static_cast<long double>(t_dur[k]) * p->fs;
    }
    p->dirty_all = true;
    p->dirty_tones.clear();
    return AWG_OK;
}

awg_status awg_update_trajectories(awg_plan *p, int64_t chunk_idx, int32_t n_upd, const int32_t *tone_idx,
                                   const double *f1, const double *t_dur, const int32_t *profile)
{
    return apply_update(p, chunk_idx, n_upd, tone_idx, f1, t_dur, profile);
}

awg_status awg_synthesize_chunk(awg_plan *p, int64_t chunk_idx, int16_t *dev_out, void *stream)
{
    awg_status st = check_chunk_call(p, chunk_idx, 1, dev_out, 16);
    if (st != AWG_OK) return st;
    return synthesize_samples(p, chunk_idx * p->chunk_len, p->chunk_len, dev_out, false, static_cast<cudaStream_t>(stream));
}

awg_status awg_synthesize_chunk_f32(awg_plan *p, int64_t chunk_idx, float *dev_out, void *stream)
{
    awg_status st = check_chunk_call(p, chunk_idx, 1, dev_out, 16);
    if (st != AWG_OK) return st;
    return synthesize_samples(p, chunk_idx * p->chunk_len, p->chunk_len, dev_out, true, static_cast<cudaStream_t>(stream));
}

awg_status awg_synthesize_range(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int16_t *dev_out, void *stream)
{
    awg_status st = check_chunk_call(p, first_chunk, n_chunks, dev_out, 16);
    if (st != AWG_OK) return st;
    return synthesize_samples(p, first_chunk * p->chunk_len, n_chunks * p->chunk_len, dev_out, false, static_cast<cudaStream_t>(stream));
}

awg_status awg_synthesize_range_host(awg_plan *p, int64_t first_chunk, int64_t n_chunks, int16_t *host_out)
{
    awg_status st = check_chunk_call(p, first_chunk, n_chunks, host_out, 2);
    if (st != AWG_OK) return st;
    cudaError_t e;
    // kE2eSlots device slots of 2^21 samples (4 MiB of int16).  Pieces alternate between two synthesis streams, so the
    // persistent CTAs of piece i+1 take over SM by SM as those of piece i run out of tiles (no idle tail between pieces),
    // while the copy stream moves finished pieces to the host.
    constexpr int64_t kPiece = int64_t(1) << 21;
    if (!p->e2e_ok) {
        awg_status bad = AWG_OK;
        for (int s = 0; s < kE2eSlots && bad == AWG_OK; ++s) {
            if ((e = cudaMalloc(reinterpret_cast<void **>(&p->e2e_slot[s]), kPiece * sizeof(int16_t))) != cudaSuccess)
                bad = fail(AWG_ERR_ALLOC, "cudaMalloc(e2e slot): %s", cudaGetErrorString(e));
            else if ((e = cudaEventCreateWithFlags(&p->e2e_ready[s], cudaEventDisableTiming)) != cudaSuccess ||
                     (e = cudaEventCreateWithFlags(&p->e2e_done[s], cudaEventDisableTiming)) != cudaSuccess)
                bad = fail_cuda(e, "e2e event creation");
        }
        for (int s = 0; s < 3 && bad == AWG_OK; ++s)
            if ((e = cudaStreamCreateWithFlags(&p->e2e_stream[s], cudaStreamNonBlocking)) != cudaSuccess)
                bad = fail_cuda(e, "e2e stream creation");
        if (bad != AWG_OK) {
            free_e2e(p);   // all or nothing: a half-built set is torn down again
            return bad;
        }
        p->e2e_ok = true;
    }
    const int64_t n0 = first_chunk * p->chunk_len, total = n_chunks * p->chunk_len;
    cudaStream_t s_cpy = p->e2e_stream[2];
    int i = 0;
    for (int64_t off = 0; off < total; off += kPiece, ++i) {
        const int slot = i % kE2eSlots;
        cudaStream_t s_syn = p->e2e_stream[i & 1];
        const int64_t cnt = (total - off < kPiece) ? (total - off) : kPiece;
        if (i >= kE2eSlots && (e = cudaStreamWaitEvent(s_syn, p->e2e_done[slot], 0)) != cudaSuccess) return fail_cuda(e, "cudaStreamWaitEvent");
        if ((st = synthesize_samples(p, n0 + off, cnt, p->e2e_slot[slot], false, s_syn)) != AWG_OK) return st;
        if ((e = cudaEventRecord(p->e2e_ready[slot], s_syn)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
        if ((e = cudaStreamWaitEvent(s_cpy, p->e2e_ready[slot], 0)) != cudaSuccess) return fail_cuda(e, "cudaStreamWaitEvent");
        if ((e = cudaMemcpyAsync(host_out + off, p->e2e_slot[slot], cnt * sizeof(int16_t), cudaMemcpyDeviceToHost, s_cpy)) != cudaSuccess)
            return fail_cuda(e, "cudaMemcpyAsync(D2H)");
        if ((e = cudaEventRecord(p->e2e_done[slot], s_cpy)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
        p->d2h_bytes += cnt * static_cast<int64_t>(sizeof(int16_t));
    }
    if ((e = cudaStreamSynchronize(s_cpy)) != cudaSuccess) return fail_cuda(e, "cudaStreamSynchronize");
    return AWG_OK;
}

}  // extern "C"
