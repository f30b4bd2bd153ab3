// pipe_rates.cu -- instruction-mix microbenchmarks behind the roofline peaks and the loop design of DESIGN.md section 6.
//
// Not part of the library (nothing links it).  Build and run on a B200:
//     nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/pipe_rates paper_2403_15582_b200/ubench/pipe_rates.cu
//     /tmp/pipe_rates [warps_per_smsp=4]
// Every body is an unrolled block of independent instructions (inline PTX, so the mix is what the line says); a warp
// runs it kIters times, `warps_per_smsp` warps share a scheduler, every SM is filled.  Printed: SM cycles (clock64, the
// slowest CTA) per body per scheduler (SMSP), i.e. the cycles one SMSP needs for one body of EVERY resident warp divided
// by the warps -- the reciprocal throughput of the mix, independent of the clock the GPU runs at.
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>

constexpr int kIters = 4096;

#define FFMA2(acc, a, b) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b))
#define HFMA2(acc, a, b) asm volatile("fma.rn.f16x2 %0, %1, %2, %0;" : "+r"(acc) : "r"(a), "r"(b))
#define FFMA(acc, a, b) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(acc) : "f"(a), "f"(b))
#define FMUL(acc, a) asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(acc) : "f"(a))
#define FMUL2(acc, a) asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(acc) : "l"(a))
#define MUFU_SIN(acc) asm volatile("sin.approx.ftz.f32 %0, %0;" : "+f"(acc))
#define MUFU_EX2(acc) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(acc))
#define IADD(acc, a) asm volatile("add.u32 %0, %0, %1;" : "+r"(acc) : "r"(a))
#define IMAD(acc, a, b) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(acc) : "r"(a), "r"(b))
#define I2F(dst, src) asm volatile("cvt.rn.f32.s32 %0, %1;" : "=f"(dst) : "r"(src))
#define LDS128(dst, addr) asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(dst.x), "=f"(dst.y), "=f"(dst.z), "=f"(dst.w) : "r"(addr))

template <int MODE>
__global__ void __launch_bounds__(128) bench(float *out, unsigned long long seed, int n_iter, unsigned long long *cycles)
{
    const long long t_begin = clock64();
    __shared__ float4 sm[64];
    if (threadIdx.x < 64) sm[threadIdx.x] = make_float4(1.f, 1.0001f, 0.9999f, 1.f);
    __syncthreads();
    unsigned long long a2[32], x2 = seed | 0x3f8000003f800000ull, y2 = 0x3a0000003a000000ull;
    unsigned h2[32], hx = 0x3c003c00u, hy = 0x10001000u;
    float f[16], fa = 1.0001f;
    unsigned u[16], ua = 3u + threadIdx.x;
    float4 t[8];
#pragma unroll
    for (int i = 0; i < 32; ++i) { a2[i] = seed + i; h2[i] = static_cast<unsigned>(seed) + i; }
#pragma unroll
    for (int i = 0; i < 16; ++i) { f[i] = 0.001f * i + threadIdx.x; u[i] = i * 7u + threadIdx.x; }
#pragma unroll
    for (int i = 0; i < 8; ++i) t[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    const unsigned sbase = static_cast<unsigned>(__cvta_generic_to_shared(sm));
#pragma unroll 1
    for (int it = 0; it < n_iter; ++it) {
        if (MODE == 0) {          // 32 FFMA2
#pragma unroll
            for (int i = 0; i < 32; ++i) FFMA2(a2[i], x2, y2);
        } else if (MODE == 1) {   // 32 HFMA2
#pragma unroll
            for (int i = 0; i < 32; ++i) HFMA2(h2[i], hx, hy);
        } else if (MODE == 2) {   // 32 FFMA2 + 32 HFMA2 interleaved
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); HFMA2(h2[i], hx, hy); }
        } else if (MODE == 3) {   // 32 FFMA2 + 16 HFMA2
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if (i & 1) HFMA2(h2[i], hx, hy); }
        } else if (MODE == 4) {   // 32 FFMA2 + 8 scalar FMUL
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 3) == 3) FMUL(f[i >> 2], fa); }
        } else if (MODE == 5) {   // 32 FFMA2 + 8 FMUL2
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 3) == 3) FMUL2(a2[i - 1], x2); }
        } else if (MODE == 6) {   // 32 FFMA2 + 8 pairs of adjacent scalar FMUL (16 FMUL)
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 3) == 3) { FMUL(f[i >> 2], fa); FMUL(f[8 + (i >> 2)], fa); } }
        } else if (MODE == 7) {   // 32 FFMA2 + 8 MUFU.EX2
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 3) == 3) MUFU_EX2(f[i >> 2]); }
        } else if (MODE == 8) {   // 32 FFMA2 + 8 sin.approx (FMUL.RZ + MUFU.SIN)
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 3) == 3) MUFU_SIN(f[i >> 2]); }
        } else if (MODE == 9) {   // 32 FFMA2 + 4 MUFU.EX2
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 7) == 7) MUFU_EX2(f[i >> 3]); }
        } else if (MODE == 10) {  // 32 FFMA2 + 5 LDS.128 broadcast
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if (i % 6 == 5) LDS128(t[i / 6], sbase + 16 * (i / 6)); }
        } else if (MODE == 11) {  // 32 FFMA2 + 9 LDS.128 broadcast
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if (i % 4 == 3) LDS128(t[i / 4], sbase + 16 * (i / 4)); }
        } else if (MODE == 12) {  // 32 FFMA2 + 16 IADD + 8 I2F
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if (i & 1) IADD(u[i >> 1], ua); if ((i & 3) == 3) I2F(f[i >> 2], u[i >> 2]); }
        } else if (MODE == 13) {  // 32 FFMA2 + 4 IMAD
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 7) == 7) IMAD(u[i >> 3], ua, ua); }
        } else if (MODE == 14) {  // 64 scalar FFMA
#pragma unroll
            for (int i = 0; i < 16; ++i) { FFMA(f[i], fa, fa); FFMA(f[i], fa, fa); FFMA(f[i], fa, fa); FFMA(f[i], fa, fa); }
        } else if (MODE == 15) {  // static-loop mix: 32 FFMA2 + 5 LDS.128 + 8 MUFU(4 sin.approx pairs ~ 4 FMUL.RZ) + 2 FMUL2 + 4 I2F + 4 IADD + 1 IMAD
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                FFMA2(a2[i], x2, y2);
                if (i % 6 == 5) LDS128(t[i / 6], sbase + 16 * (i / 6));
                if ((i & 7) == 3) MUFU_SIN(f[i >> 3]);
                if ((i & 7) == 7) MUFU_EX2(f[8 + (i >> 3)]);
                if ((i & 15) == 9) FMUL2(a2[i - 1], x2);
                if ((i & 7) == 1) { IADD(u[i >> 3], ua); I2F(f[4 + (i >> 3)], u[i >> 3]); }
                if (i == 20) IMAD(u[8], ua, ua);
            }
        } else if (MODE == 16) {  // 16 FFMA2 + 16 HFMA2 (slow-pass idea: correction in half precision)
#pragma unroll
            for (int i = 0; i < 16; ++i) { FFMA2(a2[i], x2, y2); HFMA2(h2[i], hx, hy); }
        } else if (MODE == 18) {  // 32 FFMA2 + 8 I2F
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 3) == 3) I2F(f[i >> 2], u[i >> 2]); }
        } else if (MODE == 19) {  // 32 FFMA2 + 16 LOP3 (xor)
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if (i & 1) asm volatile("xor.b32 %0, %0, %1;" : "+r"(u[i >> 1]) : "r"(ua)); }
        } else if (MODE == 20) {  // 32 FFMA2 + 4 I2F
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); if ((i & 7) == 7) I2F(f[i >> 3], u[i >> 3]); }
        } else if (MODE == 21) {  // 32 FFMA2 + 32 LOP3
#pragma unroll
            for (int i = 0; i < 32; ++i) { FFMA2(a2[i], x2, y2); asm volatile("xor.b32 %0, %0, %1;" : "+r"(u[i & 15]) : "r"(ua)); }
        } else if (MODE == 22) {  // rotation mix: 32 FFMA2 + 5 LDS.128 + 2 sin.approx + 2 MUFU.EX2 + 1 FMUL2 + 4 packed rotation ops (2 FMUL2 + 2 FFMA2) + 2 I2F
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                FFMA2(a2[i], x2, y2);
                if (i % 6 == 5) LDS128(t[i / 6], sbase + 16 * (i / 6));
                if ((i & 15) == 3) MUFU_SIN(f[i >> 4]);
                if ((i & 15) == 7) MUFU_EX2(f[8 + (i >> 4)]);
                if (i == 9) FMUL2(a2[i - 1], x2);
                if (i == 13 || i == 21) FMUL2(a2[i - 2], x2);
                if (i == 17 || i == 25) FFMA2(a2[i - 3], x2, y2);
                if ((i & 15) == 1) I2F(f[4 + (i >> 4)], u[i >> 4]);
            }
        } else if (MODE == 23) {  // slow-pass mix: 64 FFMA2 + 9 LDS.128 + 4 sin.approx + 4 MUFU.EX2 + 10 packed fp32x2 + 4 I2F
#pragma unroll
            for (int i = 0; i < 64; ++i) {
                FFMA2(a2[i & 31], x2, y2);
                if (i % 7 == 6) LDS128(t[(i / 7) & 7], sbase + 16 * (i / 7));
                if ((i & 15) == 3) MUFU_SIN(f[i >> 4]);
                if ((i & 15) == 7) MUFU_EX2(f[8 + (i >> 4)]);
                if (i % 6 == 2) FMUL2(a2[(i + 5) & 31], x2);
                if ((i & 15) == 1) I2F(f[4 + (i >> 4)], u[i >> 4]);
            }
        } else if (MODE == 17) {  // 8 MUFU.SIN alone
#pragma unroll
            for (int i = 0; i < 8; ++i) MUFU_SIN(f[i]);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 32; ++i) s += static_cast<float>(a2[i] & 0xff) + static_cast<float>(h2[i] & 0xff);
#pragma unroll
    for (int i = 0; i < 16; ++i) s += f[i] + static_cast<float>(u[i]);
#pragma unroll
    for (int i = 0; i < 8; ++i) s += t[i].x + t[i].y + t[i].z + t[i].w;
    if (s == 123.456f) out[0] = s;
    if (threadIdx.x == 0) atomicMax(cycles, static_cast<unsigned long long>(clock64() - t_begin));
}

// The multiply-add loop of the angle-addition pass as the library writes it: 4 groups x (4 P + 4 Q) packed accumulators,
// one tone's pair tables from shared memory (4 broadcast LDS.128), sines/cosines broadcast from scalar registers,
// software-pipelined one tone ahead and unrolled by two (ping-pong register sets), 3 CTAs of 128 threads per SM.
// SC = 0: the multiply-adds alone; 1: plus the round-1 chain IMAD, 3 IADD, 4 I2F, 2 FMUL2, 4 sin.approx, 4 cos.approx per
// tone; 2: the round-2 chain: two sin/cos pairs from MUFU, the other two by a packed rotation (2 FMUL2 + 2 FFMA2).
struct PQu { float2 P[4], Q[4]; };
__device__ __forceinline__ void pq_add_u(PQu &pq, float s, float c, const float4 &C03, const float4 &C47, const float4 &S03, const float4 &S47)
{
    const float2 s2 = make_float2(s, s), c2 = make_float2(c, c);
    pq.P[0] = __ffma2_rn(s2, make_float2(C03.x, C03.y), pq.P[0]);
    pq.P[1] = __ffma2_rn(s2, make_float2(C03.z, C03.w), pq.P[1]);
    pq.P[2] = __ffma2_rn(s2, make_float2(C47.x, C47.y), pq.P[2]);
    pq.P[3] = __ffma2_rn(s2, make_float2(C47.z, C47.w), pq.P[3]);
    pq.Q[0] = __ffma2_rn(c2, make_float2(S03.x, S03.y), pq.Q[0]);
    pq.Q[1] = __ffma2_rn(c2, make_float2(S03.z, S03.w), pq.Q[1]);
    pq.Q[2] = __ffma2_rn(c2, make_float2(S47.x, S47.y), pq.Q[2]);
    pq.Q[3] = __ffma2_rn(c2, make_float2(S47.z, S47.w), pq.Q[3]);
}
__device__ __forceinline__ float usin(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float ucos(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
template <int SC>
__device__ __forceinline__ void sincos4_u(const uint4 cc, const float4 rot, int off, float (&s)[4], float (&c)[4])
{
    const float k = 1.4629180792671596e-9f;
    const float2 k2 = make_float2(k, k);
    const unsigned p0 = cc.x + cc.y * static_cast<unsigned>(off), p1 = p0 + cc.z;
    const float2 x01 = __fmul2_rn(make_float2(__int2float_rn(static_cast<int>(p0)), __int2float_rn(static_cast<int>(p1))), k2);
    s[0] = usin(x01.x); c[0] = ucos(x01.x); s[1] = usin(x01.y); c[1] = ucos(x01.y);
    if (SC == 1) {
        const unsigned p2 = p1 + cc.z, p3 = p2 + cc.z;
        const float2 x23 = __fmul2_rn(make_float2(__int2float_rn(static_cast<int>(p2)), __int2float_rn(static_cast<int>(p3))), k2);
        s[2] = usin(x23.x); c[2] = ucos(x23.x); s[3] = usin(x23.y); c[3] = ucos(x23.y);
    } else {
        const float2 s01 = make_float2(s[0], s[1]), c01 = make_float2(c[0], c[1]);
        const float2 s23 = __ffma2_rn(c01, make_float2(rot.y, rot.y), __fmul2_rn(s01, make_float2(rot.x, rot.x)));
        const float2 c23 = __ffma2_rn(s01, make_float2(-rot.y, -rot.y), __fmul2_rn(c01, make_float2(rot.x, rot.x)));
        s[2] = s23.x; s[3] = s23.y; c[2] = c23.x; c[3] = c23.y;
    }
}

// staged record: 6 float4 per tone: {c0, c1, d, -}, C03, C47, S03, S47, {cos, sin of the rotation, -, -}
template <int SC>
__global__ void __launch_bounds__(128, 3) pq_loop(float *out, int n_iter, unsigned long long *cycles)
{
    const long long t_begin = clock64();
    __shared__ float4 tab[67 * 6];
    for (int i = threadIdx.x; i < 67 * 6; i += 128) tab[i] = make_float4(1e-3f * i, 1.f, 0.5f, 0.25f);
    __syncthreads();
    PQu pq[4];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int m = 0; m < 4; ++m) pq[r].P[m] = pq[r].Q[m] = make_float2(0.f, 0.f);
    const int off = (threadIdx.x & 31) - 16;
    float sa[4] = {0.1f, 0.2f, 0.3f, 0.4f}, ca[4] = {0.9f, 0.8f, 0.7f, 0.6f}, sb[4] = {0.11f, 0.21f, 0.31f, 0.41f}, cb[4] = {0.89f, 0.79f, 0.69f, 0.59f};
    for (int it = 0; it < n_iter; it += 64) {
        const float4 *sp = tab;
        if (SC) sincos4_u<SC ? SC : 1>(*reinterpret_cast<const uint4 *>(sp), sp[5], off, sa, ca);
#pragma unroll 1
        for (int i = 0; i < 64; i += 2, sp += 12) {
            {
                const float4 C03 = sp[1], C47 = sp[2], S03 = sp[3], S47 = sp[4];
                if (SC) sincos4_u<SC ? SC : 1>(*reinterpret_cast<const uint4 *>(sp + 6), sp[11], off, sb, cb);
#pragma unroll
                for (int r = 0; r < 4; ++r) pq_add_u(pq[r], sa[r], ca[r], C03, C47, S03, S47);
            }
            {
                const float4 C03 = sp[7], C47 = sp[8], S03 = sp[9], S47 = sp[10];
                if (SC) sincos4_u<SC ? SC : 1>(*reinterpret_cast<const uint4 *>(sp + 12), sp[17], off, sa, ca);
#pragma unroll
                for (int r = 0; r < 4; ++r) pq_add_u(pq[r], sb[r], cb[r], C03, C47, S03, S47);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int m = 0; m < 4; ++m) s += pq[r].P[m].x + pq[r].P[m].y + pq[r].Q[m].x + pq[r].Q[m].y;
    if (s == 123.456f) out[0] = s;
    if (threadIdx.x == 0) atomicMax(cycles, static_cast<unsigned long long>(clock64() - t_begin));
}

template <int SC>
void run_pq(const char *what, int n_sm, int wps, float *out)
{
    unsigned long long *cyc_dev, cyc_host = 0;
    cudaMalloc(&cyc_dev, sizeof cyc_host);
    pq_loop<SC><<<n_sm * wps, 128>>>(out, 64, cyc_dev);
    cudaMemset(cyc_dev, 0, sizeof cyc_host);
    pq_loop<SC><<<n_sm * wps, 128>>>(out, kIters, cyc_dev);
    cudaMemcpy(&cyc_host, cyc_dev, sizeof cyc_host, cudaMemcpyDeviceToHost);
    cudaFree(cyc_dev);
    printf("%-100s %8.2f cycles/body/SMSP\n", what, static_cast<double>(cyc_host) / (static_cast<double>(kIters) * wps));
}

template <int MODE>
void run(const char *what, int n_sm, int wps, double mhz, float *out)
{
    const int ctas = n_sm * wps;  // 4 warps per CTA: one per scheduler
    unsigned long long *cyc_dev, cyc_host = 0;
    cudaMalloc(&cyc_dev, sizeof cyc_host);
    bench<MODE><<<ctas, 128>>>(out, 1ull, 64, cyc_dev);
    cudaMemset(cyc_dev, 0, sizeof cyc_host);
    bench<MODE><<<ctas, 128>>>(out, 1ull, kIters, cyc_dev);
    cudaMemcpy(&cyc_host, cyc_dev, sizeof cyc_host, cudaMemcpyDeviceToHost);
    cudaFree(cyc_dev);
    (void)mhz;
    // SM cycles (clock64) of the slowest CTA: independent of the clock the GPU happens to run at
    printf("%-100s %8.2f cycles/body/SMSP\n", what, static_cast<double>(cyc_host) / (static_cast<double>(kIters) * wps));
}

int main(int argc, char **argv)
{
    const int wps = argc > 1 ? atoi(argv[1]) : 4;
    cudaDeviceProp pr;
    cudaGetDeviceProperties(&pr, 0);
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    const double mhz = khz / 1e3;
    float *out;
    cudaMalloc(&out, 64);
    printf("%s, %d SMs, %.0f MHz (max SM clock), %d warps per SMSP\n", pr.name, pr.multiProcessorCount, mhz, wps);
    const int n = pr.multiProcessorCount;
    run<0>("32 FFMA2", n, wps, mhz, out);
    run<1>("32 HFMA2", n, wps, mhz, out);
    run<2>("32 FFMA2 + 32 HFMA2", n, wps, mhz, out);
    run<3>("32 FFMA2 + 16 HFMA2", n, wps, mhz, out);
    run<16>("16 FFMA2 + 16 HFMA2", n, wps, mhz, out);
    run<4>("32 FFMA2 + 8 FMUL (scalar)", n, wps, mhz, out);
    run<5>("32 FFMA2 + 8 FMUL2", n, wps, mhz, out);
    run<6>("32 FFMA2 + 8 x 2 adjacent scalar FMUL", n, wps, mhz, out);
    run<7>("32 FFMA2 + 8 MUFU.EX2", n, wps, mhz, out);
    run<8>("32 FFMA2 + 8 sin.approx (FMUL.RZ + MUFU.SIN)", n, wps, mhz, out);
    run<9>("32 FFMA2 + 4 MUFU.EX2", n, wps, mhz, out);
    run<10>("32 FFMA2 + 5 LDS.128 (broadcast)", n, wps, mhz, out);
    run<11>("32 FFMA2 + 8 LDS.128 (broadcast)", n, wps, mhz, out);
    run<12>("32 FFMA2 + 16 IADD + 8 I2F", n, wps, mhz, out);
    run<13>("32 FFMA2 + 4 IMAD", n, wps, mhz, out);
    run<14>("64 FFMA (scalar)", n, wps, mhz, out);
    run<15>("static-loop mix: 32 FFMA2 + 5 LDS.128 + 4 sin.approx + 4 MUFU.EX2 + 2 FMUL2 + 4 IADD + 4 I2F + 1 IMAD", n, wps, mhz, out);
    run<17>("8 sin.approx", n, wps, mhz, out);
    run<18>("32 FFMA2 + 8 I2F", n, wps, mhz, out);
    run<20>("32 FFMA2 + 4 I2F", n, wps, mhz, out);
    run<19>("32 FFMA2 + 16 LOP3", n, wps, mhz, out);
    run<21>("32 FFMA2 + 32 LOP3", n, wps, mhz, out);
    run<22>("rotation mix: 32 FFMA2 + 5 LDS.128 + 2 sin.approx + 2 MUFU.EX2 + 3 FMUL2 + 2 more FFMA2 + 2 I2F", n, wps, mhz, out);
    run<23>("slow-pass mix: 64 FFMA2 + 9 LDS.128 + 4 sin.approx + 4 MUFU.EX2 + 11 FMUL2 + 4 I2F", n, wps, mhz, out);
    run_pq<0>("library multiply-add loop (body = one tone): 32 FFMA2, distinct accumulators, tables from 4 LDS.128, broadcast sines", n, wps, out);
    run_pq<1>("library static loop, round 1: the same + IMAD, 3 IADD, 4 I2F, 2 FMUL2, 4 sin.approx, 4 cos.approx per tone", n, wps, out);
    run_pq<2>("library static loop, round 2: IMAD, IADD, 2 I2F, FMUL2, 2 sin.approx, 2 cos.approx + packed rotation (2 FMUL2, 2 FFMA2)", n, wps, out);
    return 0;
}
