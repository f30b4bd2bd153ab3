/* ORACLE -- test infrastructure, not product code.
 *
 * Plain C evaluator of the additive-synthesis definition of arXiv 2403.15582, written
 * independently of (and sharing no code with) the CUDA path.  Same definition as
 * oracle/awg_oracle.py, one sample at a time, one libm sin() per (tone, sample), phases in
 * x87 long double (64-bit mantissa), sum over tones in double in tone order.  No tiling,
 * no recurrences, no tables.  It exists because the numpy version is too slow for the
 * 10^8..10^10 tone-sample configurations; tests/test_oracle_pins.py checks the two against
 * each other and both against closed forms.  It is also the timed "cpu_baseline" of bench.py,
 * as it stands (it is never tuned for that).
 *
 * Per (tone k, absolute sample n), t = n/fs, tau = t - t_s, D = f1 - f0 (PAPER.md:<line>):
 *   STATIC or tau <= 0 :  Phi = theta + f0 t                               Eq. 8
 *   LINEAR  0<tau<T    :  Phi = theta + f0 t + D T s^2/2 ,  s = tau/T      named at PAPER.md:137
 *   MINJERK 0<tau<T    :  Phi = theta + f0 t + D T (5/2 s^4 - 3 s^5 + s^6) Eq. 10 / p(i), PAPER.md:141-148,
 *                                                                          prefactor corrected to T (G1)
 *   tau >= T           :  Phi = theta + f0 t_s + f1 tau + T (f0 - f1)/2    Eq. 10 branch 2
 *   V[n] = sum_k a_k[n] sin(2 pi frac(Phi_k[n]))                           Eq. 9, Eq. 14
 *   a_k[n] = A_k, or with an amplitude ramp (awg_oracle_waveform_amp; Eq. 9 allows a_j[i], reading G7 in DESIGN.md):
 *            A_k before t_a, A_k + (A1_k - A_k) h((t - t_a)/T_a) during it, A1_k after; h(s) = s or 10 s^3 - 15 s^4 + 6 s^5
 *   code = clamp(rint(scale V), -32768, 32767)                             PAPER.md:77, 196; G9
 *
 * Segment table layout (built by OraclePlan.flat_segments): tone k owns segments
 * seg_off[k] .. seg_off[k+1]-1 in time order; seg_n_begin[i] is the first absolute sample
 * segment i applies to (a very negative number for a tone's first segment);
 * reals is 5 rows (t_s, T, f0, f1, theta[cycles]) of S long doubles each.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define AWG_STATIC 0
#define AWG_LINEAR 1
#define AWG_MINJERK 2
#define AWG_EXP 3   /* exponential chirp f0 (f1/f0)^(tau/T), named at PAPER.md:137 (reading G20) */

static long double seg_phase(long double t, long double t_s, long double T, long double f0,
                             long double f1, long double theta, int profile)
{
    long double tau = t - t_s;
    if (profile == AWG_STATIC || tau <= 0.0L)
        return theta + f0 * t;
    if (profile == AWG_EXP) {
        /* phase gained since the start of the move: f0 T (r^s - 1)/ln r, r = f1/f0; T (f1 - f0)/ln r over the whole move */
        if (f1 == f0 || !(T > 0.0L)) {
            if (tau >= T) return theta + f0 * t_s + f0 * T + f1 * (tau - T);
            return theta + f0 * t;
        }
        long double Lr = logl(f1 / f0);
        if (tau >= T) return theta + f0 * t_s + T * (f1 - f0) / Lr + f1 * (tau - T);
        return theta + f0 * t_s + f0 * T * expm1l(Lr * (tau / T)) / Lr;
    }
    if (tau >= T)
        return theta + f0 * t_s + f1 * tau + T * (f0 - f1) / 2.0L;
    long double s = tau / T;
    long double g;
    if (profile == AWG_LINEAR) {
        g = s * s / 2.0L;
    } else {
        long double s2 = s * s, s4 = s2 * s2;
        g = 2.5L * s4 - 3.0L * s4 * s + s4 * s2;
    }
    return theta + f0 * t + (f1 - f0) * T * g;
}

static double amp_at(long double t, double A0, double A1, double t_a, double T_a, int prof)
{
    if (prof == AWG_STATIC) return A0;
    long double tau = t - (long double)t_a;
    double s;
    if (T_a > 0.0) {
        s = (double)(tau / (long double)T_a);
        if (s < 0.0) s = 0.0;
        if (s > 1.0) s = 1.0;
    } else {
        s = tau >= 0.0L ? 1.0 : 0.0;
    }
    double h = prof == AWG_LINEAR ? s : s * s * s * (10.0 + s * (6.0 * s - 15.0));
    return A0 + (A1 - A0) * h;
}

/* V_out[n - n0] for n in [n0, n1), with optional amplitude ramps (amp_A1 == NULL: constant amplitudes).
 * Returns 0, or -1 on bad arguments. */
int awg_oracle_waveform_amp(int32_t n_tones, double fs, const int64_t *seg_off, const int64_t *seg_n_begin,
                            const long double *reals, int64_t n_segs, const int32_t *profile,
                            const double *A, const double *amp_A1, const double *amp_ts, const double *amp_T,
                            const int32_t *amp_prof, int64_t n0, int64_t n1, double *V_out, int32_t n_threads)
{
    if (n_tones < 1 || !(fs > 0.0) || !seg_off || !seg_n_begin || !reals || !profile || !A || !V_out || n1 < n0)
        return -1;
    if (amp_A1 && (!amp_ts || !amp_T || !amp_prof)) return -1;
    const long double *t_s = reals, *T = reals + n_segs, *f0 = reals + 2 * n_segs,
                      *f1 = reals + 3 * n_segs, *theta = reals + 4 * n_segs;
    const long double fsl = (long double)fs;
    const double two_pi = 6.283185307179586476925286766559;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(static)
    for (int64_t n = n0; n < n1; ++n) {
        long double t = (long double)n / fsl;
        double v = 0.0;
        for (int32_t k = 0; k < n_tones; ++k) {
            /* last segment of tone k whose n_begin <= n */
            int64_t lo = seg_off[k], hi = seg_off[k + 1] - 1;
            while (lo < hi) {
                int64_t mid = (lo + hi + 1) / 2;
                if (seg_n_begin[mid] <= n) lo = mid; else hi = mid - 1;
            }
            long double ph = seg_phase(t, t_s[lo], T[lo], f0[lo], f1[lo], theta[lo], profile[lo]);
            long double fr = ph - floorl(ph);
            double a = amp_A1 ? amp_at(t, A[k], amp_A1[k], amp_ts[k], amp_T[k], amp_prof[k]) : A[k];
            v += a * sin(two_pi * (double)fr);
        }
        V_out[n - n0] = v;
    }
    return 0;
}

int awg_oracle_waveform(int32_t n_tones, double fs, const int64_t *seg_off, const int64_t *seg_n_begin,
                        const long double *reals, int64_t n_segs, const int32_t *profile,
                        const double *A, int64_t n0, int64_t n1, double *V_out, int32_t n_threads)
{
    return awg_oracle_waveform_amp(n_tones, fs, seg_off, seg_n_begin, reals, n_segs, profile, A, NULL, NULL, NULL, NULL,
                                   n0, n1, V_out, n_threads);
}

int awg_oracle_quantise(const double *V, int64_t n, double scale, int16_t *out)
{
    if (!V || !out || n < 0) return -1;
    for (int64_t i = 0; i < n; ++i) {
        double q = rint(scale * V[i]); /* default rounding mode: half to even */
        if (q > 32767.0) q = 32767.0;
        if (q < -32768.0) q = -32768.0;
        out[i] = (int16_t)q;
    }
    return 0;
}

int awg_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
