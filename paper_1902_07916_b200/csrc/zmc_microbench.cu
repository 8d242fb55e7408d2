/*
 * zmc_microbench.cu -- issue-rate microbenchmarks of the pipes the sampling kernel uses.
 * They give the denominator of the ALU roofline: the path is bound by the
 * warp schedulers' issue slots and the integer pipes (Philox is 20 IMAD.WIDE.U32 + 20 LOP3 per
 * call), not by HBM, the tensor cores or the SFU, so the peak has to come from measured
 * instruction throughput, not from a data sheet.
 *
 * Each kernel runs a long unrolled loop of the instruction under test on ILP independent chains
 * per thread, 4 CTAs of 256 threads per SM (8 warps per scheduler, one wave), and reports
 * warp-instructions / SM / clock with the clock taken from clock64() on every SM.
 */
#include <cuda_runtime.h>

#include "../../include/zmc.h"
#include "zmc_device.cuh"

namespace {

constexpr int kIters = 4096;
constexpr int kIlp = 8;

template <int WHICH>
__global__ void __launch_bounds__(256, 4) mb_kernel(zu32* sink, unsigned long long* cycles, zu32 seed) {
    const long long t0 = clock64();
    zu32 r[kIlp];
    float f[kIlp];
    double d[kIlp];
#pragma unroll
    for (int i = 0; i < kIlp; ++i) {
        r[i] = seed + threadIdx.x * 977u + i * 131u;
        f[i] = __uint_as_float(0x3f800000u | (r[i] & 0xFFFFu));
        d[i] = (double)f[i];
    }
    zu32 acc = 0;
    const zu32 k0 = seed * 3u + 1u, k1 = seed * 5u + 7u;
    const float fc = __uint_as_float(0x3f7ff000u | (seed & 0xFFu));
    const double dc = (double)fc;
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < kIlp; ++i) {
            if (WHICH == 0) {            /* IMAD.WIDE.U32: 32x32 -> 64, both halves consumed by the next one */
                const zu64 p = (zu64)r[i] * (zu64)ZMC_PHILOX_M0;
                zu32 lo, hi;
                asm volatile("mov.b64 {%0,%1}, %2;" : "=r"(lo), "=r"(hi) : "l"(p));
                asm volatile("" : "+r"(lo), "+r"(hi));
                r[i] = hi;
                acc += 0;   /* lo is dead on purpose: one instruction per step */
                (void)lo;
            } else if (WHICH == 1) {     /* LOP3 (3-input xor) */
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[i]) : "r"(k0), "r"(k1));
            } else if (WHICH == 2) {     /* Philox round mix: IMAD.WIDE.U32 + LOP3 */
                const zu64 p = (zu64)r[i] * (zu64)ZMC_PHILOX_M0;
                const zu32 lo = (zu32)p, hi = (zu32)(p >> 32);
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r[i]) : "r"(hi), "r"(lo), "r"(k0));
            } else if (WHICH == 3) {     /* FFMA */
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(fc), "f"(f[(i + 1) % kIlp]));
            } else if (WHICH == 4) {     /* FADD */
                asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(fc));
            } else if (WHICH == 5) {     /* DADD */
                asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(dc));
            } else if (WHICH == 6) {     /* F2F.F64.F32 + F2F.F32.F64 as a dependent pair (one alone is hoisted by the compiler) */
                asm volatile("{ .reg .f64 t; cvt.f64.f32 t, %0; cvt.rn.f32.f64 %0, t; }" : "+f"(f[i]));
            } else if (WHICH == 7) {     /* MUFU.SIN */
                asm volatile("sin.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
            } else if (WHICH == 8) {     /* MUFU.EX2 */
                asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
            } else if (WHICH == 9) {     /* DFMA */
                asm volatile("fma.rn.f64 %0, %0, %1, %1;" : "+d"(d[i]) : "d"(dc));
            } else if (WHICH == 11) {    /* I2F.F64.U32 + F2I.U32.F64 as a dependent pair */
                asm volatile("{ .reg .f64 t; cvt.rn.f64.u32 t, %0; cvt.rzi.u32.f64 %0, t; }" : "+r"(r[i]));
            } else if (WHICH == 12) {    /* LEA.HI-like: (w >> 9) | 0x3F800000 */
                asm volatile("{ .reg .b32 t; shr.u32 t, %0, 9; or.b32 %0, t, 0x3F800000; }" : "+r"(r[i]));
            } else if (WHICH == 13) {    /* IMAD (low 32 bits of a 32x32 product, plus an addend) */
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(k0), "r"(k1));
            } else if (WHICH == 14) {    /* IMAD.HI.U32 */
                asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(r[i]) : "r"(k0));
            } else if (WHICH == 15) {    /* 64-bit add: IADD3 + IADD3.X (counted as one) */
                asm volatile("{ add.cc.u32 %0, %0, %2; addc.u32 %1, %1, %3; }"
                             : "+r"(r[i]), "+r"(r[(i + 1) % kIlp]) : "r"(k0), "r"(k1));
            } else if (WHICH == 16) {    /* IMAD.WIDE.U32 with a register (not immediate) multiplier */
                zu32 lo, hi;
                asm volatile("{ .reg .b64 t; mul.wide.u32 t, %2, %3; mov.b64 {%0,%1}, t; }" : "=r"(lo), "=r"(hi) : "r"(r[i]), "r"(k0));
                r[i] = hi ^ 0u;
                (void)lo;
            }
        }
        if (WHICH == 10) {               /* whole Philox4x32-10 calls, kIlp/2 independent calls per step */
            ZmcKeySchedule ks;
            ks.init(k0, k1);
#pragma unroll
            for (int i = 0; i < kIlp / 2; ++i) {
                zu32 w[4];
                zmc_philox(r[i] + (zu32)it, r[i + 1], k0, k1, ks, w);
                r[i] ^= w[0] ^ w[1] ^ w[2] ^ w[3];
            }
        }
    }
#pragma unroll
    for (int i = 0; i < kIlp; ++i) acc ^= r[i] ^ __float_as_uint(f[i]) ^ (zu32)__double2loint(d[i]) ^ (zu32)__double2hiint(d[i]);
    const long long t1 = clock64();
    if (acc == 0x12345678u) sink[0] = acc;
    if (threadIdx.x == 0) atomicMax(cycles, (unsigned long long)(t1 - t0));
}

template <int W>
cudaError_t launch(int grid, zu32* sink, unsigned long long* cyc, cudaStream_t st) {
    mb_kernel<W><<<grid, 256, 0, st>>>(sink, cyc, 12345u);
    return cudaGetLastError();
}

/* Philox4x32-10 calls with K extra independent instructions of kind X after each call: the slope of
 * clocks-per-call against K is what one more instruction of that kind costs next to the generator
 * (the dispatch-slot model). 4 independent calls per thread, 8 warps per scheduler.
 * X: 1 LOP3, 2 FFMA, 3 FADD, 4 DADD, 5 FFMA2, 6 IMAD (lo), 7 SHF */
template <int X, int K>
__global__ void __launch_bounds__(256, 4) mbx_kernel(zu32* sink, unsigned long long* cycles, zu32 seed) {
    zu32 r[8];
    float f[8];
    zu64 d[8];
    double x[8];
    const zu32 k0 = seed * 3u + 1u, k1 = seed * 5u + 7u;
    const float fc = __uint_as_float(0x3f7ff000u | (seed & 0xFFu)), fd = fc * 0.5f;
    const zu64 dc = ((zu64)__float_as_uint(fc) << 32) | __float_as_uint(fc), dd = dc ^ 0x0000100000001000ull;
    const double xc = (double)fc;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        r[i] = seed + threadIdx.x * 977u + i * 131u;
        f[i] = __uint_as_float(0x3f800000u | (r[i] & 0xFFFFu));
        d[i] = ((zu64)__float_as_uint(f[i]) << 32) | __float_as_uint(f[i]);
        x[i] = f[i];
    }
    ZmcKeySchedule ks;
    ks.init(k0, k1);
    zu32 c[4][4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { c[j][0] = r[j]; c[j][1] = r[j + 4]; c[j][2] = k0 + j; c[j][3] = k1 + j; }
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters / 4; ++it) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            zu32 w[4];
            zmc_philox(c[j][0] + (zu32)it, c[j][1], c[j][2], c[j][3], ks, w);
            c[j][0] = w[0]; c[j][1] = w[1]; c[j][2] = w[2]; c[j][3] = w[3];
#pragma unroll
            for (int e = 0; e < K; ++e) {
                const int i = e & 7;
                if (X == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[i]) : "r"(k0), "r"(k1));
                if (X == 2) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(fc), "f"(fd));
                if (X == 3) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(fc));
                if (X == 4) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(x[i]) : "d"(xc));
                if (X == 5) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(d[i]) : "l"(dc), "l"(dd));
                if (X == 6) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(k0), "r"(k1));
                if (X == 7) asm volatile("shf.l.wrap.b32 %0, %0, %1, 9;" : "+r"(r[i]) : "r"(k0));
            }
        }
    }
    const long long t1 = clock64();
    zu32 acc = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc ^= r[i] ^ __float_as_uint(f[i]) ^ (zu32)d[i] ^ (zu32)(d[i] >> 32) ^ (zu32)__double2loint(x[i]);
#pragma unroll
    for (int j = 0; j < 4; ++j) acc ^= c[j][0] ^ c[j][1] ^ c[j][2] ^ c[j][3];
    if (acc == 0x12345678u) sink[0] = acc;
    if (threadIdx.x == 0) atomicMax(cycles, (unsigned long long)(t1 - t0));
}

template <int X, int K>
cudaError_t launchx(int grid, zu32* sink, unsigned long long* cyc, cudaStream_t st) {
    mbx_kernel<X, K><<<grid, 256, 0, st>>>(sink, cyc, 12345u);
    return cudaGetLastError();
}

template <int X>
cudaError_t launchx_k(int kidx, int grid, zu32* sink, unsigned long long* cyc, cudaStream_t st) {
    switch (kidx) {
        case 0: return launchx<X, 0>(grid, sink, cyc, st);
        case 1: return launchx<X, 10>(grid, sink, cyc, st);
        case 2: return launchx<X, 20>(grid, sink, cyc, st);
        case 3: return launchx<X, 40>(grid, sink, cyc, st);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_mix(int which, int grid, zu32* sink, unsigned long long* cyc, cudaStream_t st) {
    const int X = (which - 100) / 10, kidx = (which - 100) % 10;
    switch (X) {
        case 1: return launchx_k<1>(kidx, grid, sink, cyc, st);
        case 2: return launchx_k<2>(kidx, grid, sink, cyc, st);
        case 3: return launchx_k<3>(kidx, grid, sink, cyc, st);
        case 4: return launchx_k<4>(kidx, grid, sink, cyc, st);
        case 5: return launchx_k<5>(kidx, grid, sink, cyc, st);
        case 6: return launchx_k<6>(kidx, grid, sink, cyc, st);
        case 7: return launchx_k<7>(kidx, grid, sink, cyc, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace

extern "C" int zmc_microbench(int which, void* stream, double* per_sm_clk, double* sm_mhz) {
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return ZMC_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return ZMC_ERR_CUDA;
    const int grid = sms * 4;
    zu32* sink = nullptr;
    unsigned long long* cyc = nullptr;
    if (cudaMalloc(&sink, 256) != cudaSuccess || cudaMalloc(&cyc, 8) != cudaSuccess) return ZMC_ERR_CUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaError_t e = cudaSuccess;
    float ms = 0.f;
    unsigned long long hc = 0;
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {   /* the last repetition is the measurement */
        cudaMemsetAsync(cyc, 0, 8, st);
        cudaEventRecord(e0, st);
        switch (which) {
            case 0: e = launch<0>(grid, sink, cyc, st); break;
            case 1: e = launch<1>(grid, sink, cyc, st); break;
            case 2: e = launch<2>(grid, sink, cyc, st); break;
            case 3: e = launch<3>(grid, sink, cyc, st); break;
            case 4: e = launch<4>(grid, sink, cyc, st); break;
            case 5: e = launch<5>(grid, sink, cyc, st); break;
            case 6: e = launch<6>(grid, sink, cyc, st); break;
            case 7: e = launch<7>(grid, sink, cyc, st); break;
            case 8: e = launch<8>(grid, sink, cyc, st); break;
            case 9: e = launch<9>(grid, sink, cyc, st); break;
            case 10: e = launch<10>(grid, sink, cyc, st); break;
            case 11: e = launch<11>(grid, sink, cyc, st); break;
            case 12: e = launch<12>(grid, sink, cyc, st); break;
            case 13: e = launch<13>(grid, sink, cyc, st); break;
            case 14: e = launch<14>(grid, sink, cyc, st); break;
            case 15: e = launch<15>(grid, sink, cyc, st); break;
            case 16: e = launch<16>(grid, sink, cyc, st); break;
            default: e = (which >= 100 && which < 180) ? launch_mix(which, grid, sink, cyc, st) : cudaErrorInvalidValue;
        }
        cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess) e = cudaMemcpy(&hc, cyc, 8, cudaMemcpyDeviceToHost);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(cyc);
    if (e != cudaSuccess) return e == cudaErrorInvalidValue ? ZMC_ERR_ARG : ZMC_ERR_CUDA;
    /* per thread: kIters * kIlp instructions (which 2: 2 each ; which 10: kIlp/2 Philox calls per step) */
    double per_thread = (double)kIters * kIlp;
    if (which == 2 || which == 6 || which == 11) per_thread *= 2.0;
    if (which == 10) per_thread = (double)kIters * (kIlp / 2);
    if (which >= 100) per_thread = (double)(kIters / 4) * 4.0;   /* Philox calls */
    const double warps_per_sm = 4.0 * 256.0 / 32.0;
    /* all CTAs of an SM are resident at once (4 x 256 threads), so the SM's elapsed clocks ~ the longest CTA */
    if (per_sm_clk) *per_sm_clk = per_thread * warps_per_sm / (double)hc;
    if (sm_mhz) *sm_mhz = (double)hc / (ms * 1e3);
    return ZMC_OK;
}
