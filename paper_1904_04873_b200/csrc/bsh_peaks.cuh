// bsh_peaks.cuh -- on-chip peak rates of the device the context runs on, MEASURED ("to be
// measured on the box with a conflict-free shared-memory load microbenchmark ... measured DADD/DMUL rate").  These are
// the denominators of the roofline fractions bench.py reports for the stage-1 accumulation kernels, which are bound on
// chip (instruction issue, FP32-add pipe, shared-memory wavefronts), not by HBM.
//
// Every kernel runs 32 warps per SM on every SM, times its unrolled body with clock64() per block, and reports
// operations per SM clock; bsh_measure_peaks() also measures the SM clock itself (clock64 against globaltimer) so that
// rates per second follow.  Bodies are volatile inline PTX: ptxas can neither delete nor fuse them.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bsh {

constexpr int kPeakThreads = 1024;    // one block of 32 warps per SM: 8 warps per scheduler
constexpr int kPeakUnroll = 256;      // operations per thread per loop iteration (loop overhead: ~1 %)

enum PeakOp { kOpLop3 = 0, kOpFadd, kOpDadd, kOpDmul, kOpMixed, kOpLds32, kOpLds64, kOpLds128, kOpCount };

struct PeakSample {
    long long cycles;                 // clock64 delta of the block (SM clocks)
    unsigned long long ns;            // globaltimer delta of the block
};

#define BSH_REP8(X) X X X X X X X X X X X X X X X X X X X X X X X X X X X X X X X X   /* 32 x 8 operations */

template <int OP>
__global__ void __launch_bounds__(kPeakThreads, 1) peak_kernel(int iters, uint32_t seed, uint32_t *sink, PeakSample *samples)
{
    __shared__ __align__(16) uint32_t sm[kPeakThreads * 8];
    for (int i = threadIdx.x; i < kPeakThreads * 8; i += blockDim.x) sm[i] = i * 2654435761u + seed;
    __syncthreads();
    uint32_t r0 = threadIdx.x + seed, r1 = r0 * 3u, r2 = r0 * 5u, r3 = r0 * 7u, r4 = r0 * 11u, r5 = r0 * 13u, r6 = r0 * 17u, r7 = r0 * 19u;
    float f0 = 1.f + r0 * 1e-9f, f1 = f0 + 1.f, f2 = f0 + 2.f, f3 = f0 + 3.f, f4 = f0 + 4.f, f5 = f0 + 5.f, f6 = f0 + 6.f, f7 = f0 + 7.f;
    double d0 = 1.0 + r0 * 1e-12, d1 = d0 + 1.0, d2 = d0 + 2.0, d3 = d0 + 3.0, d4 = d0 + 4.0, d5 = d0 + 5.0, d6 = d0 + 6.0, d7 = d0 + 7.0;
    const float fw = 1e-30f * (float)(seed & 3u);
    const double dw = 1e-300 * (double)(seed & 3u), dm = 1.0 + 1e-16 * (double)(seed & 3u);
    const uint32_t pred_src = seed | 1u;                 // always-true predicate the compiler cannot see through
    const uint32_t a4 = (uint32_t)__cvta_generic_to_shared(sm) + threadIdx.x * 4u;     // conflict-free lane addresses
    const uint32_t a8 = (uint32_t)__cvta_generic_to_shared(sm) + threadIdx.x * 8u;
    const uint32_t a16 = (uint32_t)__cvta_generic_to_shared(sm) + threadIdx.x * 16u;
    uint32_t l0 = 0, l1 = 0, l2 = 0, l3 = 0;
    unsigned long long ns0, ns1;
    __syncthreads();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns0));
    const long long c0 = clock64();
    for (int it = 0; it < iters; ++it) {
        if (OP == kOpLop3) {
            BSH_REP8(asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;\n\tlop3.b32 %1, %1, %2, %3, 0x96;\n\t"
                                  "lop3.b32 %2, %2, %3, %4, 0x96;\n\tlop3.b32 %3, %3, %4, %5, 0x96;\n\t"
                                  "lop3.b32 %4, %4, %5, %6, 0x96;\n\tlop3.b32 %5, %5, %6, %7, 0x96;\n\t"
                                  "lop3.b32 %6, %6, %7, %0, 0x96;\n\tlop3.b32 %7, %7, %0, %1, 0x96;"
                                  : "+r"(r0), "+r"(r1), "+r"(r2), "+r"(r3), "+r"(r4), "+r"(r5), "+r"(r6), "+r"(r7));)
        } else if (OP == kOpFadd) {
            // the weighted number count's inner operation: an FP32 add under a predicate (Eq. 22)
            BSH_REP8(asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %9, 0;\n\t"
                                  "@p add.f32 %0, %0, %8;\n\t@p add.f32 %1, %1, %8;\n\t@p add.f32 %2, %2, %8;\n\t"
                                  "@p add.f32 %3, %3, %8;\n\t@p add.f32 %4, %4, %8;\n\t@p add.f32 %5, %5, %8;\n\t"
                                  "@p add.f32 %6, %6, %8;\n\t@p add.f32 %7, %7, %8;\n\t}"
                                  : "+f"(f0), "+f"(f1), "+f"(f2), "+f"(f3), "+f"(f4), "+f"(f5), "+f"(f6), "+f"(f7)
                                  : "f"(fw), "r"(pred_src));)
        } else if (OP == kOpDadd) {
            BSH_REP8(asm volatile("add.rn.f64 %0, %0, %8;\n\tadd.rn.f64 %1, %1, %8;\n\tadd.rn.f64 %2, %2, %8;\n\t"
                                  "add.rn.f64 %3, %3, %8;\n\tadd.rn.f64 %4, %4, %8;\n\tadd.rn.f64 %5, %5, %8;\n\t"
                                  "add.rn.f64 %6, %6, %8;\n\tadd.rn.f64 %7, %7, %8;"
                                  : "+d"(d0), "+d"(d1), "+d"(d2), "+d"(d3), "+d"(d4), "+d"(d5), "+d"(d6), "+d"(d7)
                                  : "d"(dw));)
        } else if (OP == kOpDmul) {
            BSH_REP8(asm volatile("mul.rn.f64 %0, %0, %8;\n\tmul.rn.f64 %1, %1, %8;\n\tmul.rn.f64 %2, %2, %8;\n\t"
                                  "mul.rn.f64 %3, %3, %8;\n\tmul.rn.f64 %4, %4, %8;\n\tmul.rn.f64 %5, %5, %8;\n\t"
                                  "mul.rn.f64 %6, %6, %8;\n\tmul.rn.f64 %7, %7, %8;"
                                  : "+d"(d0), "+d"(d1), "+d"(d2), "+d"(d3), "+d"(d4), "+d"(d5), "+d"(d6), "+d"(d7)
                                  : "d"(dm));)
        } else if (OP == kOpMixed) {
            // issue-rate probe: one integer-ALU instruction per three FP32 adds, so that neither pipe alone is the limit
            // (the ALU pipe takes a warp instruction every other clock, the FP32 pipe one per clock)
            BSH_REP8(asm volatile("lop3.b32 %0, %0, %1, %0, 0x96;\n\tadd.f32 %2, %2, %8;\n\tadd.f32 %3, %3, %8;\n\t"
                                  "add.f32 %4, %4, %8;\n\tlop3.b32 %1, %1, %0, %1, 0x96;\n\tadd.f32 %5, %5, %8;\n\t"
                                  "add.f32 %6, %6, %8;\n\tadd.f32 %7, %7, %8;"
                                  : "+r"(r0), "+r"(r1), "+f"(f2), "+f"(f3), "+f"(f4), "+f"(f5), "+f"(f6), "+f"(f7)
                                  : "f"(fw));)
        } else if (OP == kOpLds32) {
            // every loaded word is consumed (3-input XOR into four chains), so no load can be dropped or merged
            BSH_REP8(asm volatile("{\n\t.reg .b32 t<8>;\n\t"
                                  "ld.volatile.shared.u32 t0, [%4];\n\tld.volatile.shared.u32 t1, [%4+4096];\n\t"
                                  "ld.volatile.shared.u32 t2, [%4+8192];\n\tld.volatile.shared.u32 t3, [%4+12288];\n\t"
                                  "ld.volatile.shared.u32 t4, [%4+16384];\n\tld.volatile.shared.u32 t5, [%4+20480];\n\t"
                                  "ld.volatile.shared.u32 t6, [%4+24576];\n\tld.volatile.shared.u32 t7, [%4+28672];\n\t"
                                  "lop3.b32 %0, %0, t0, t1, 0x96;\n\tlop3.b32 %1, %1, t2, t3, 0x96;\n\t"
                                  "lop3.b32 %2, %2, t4, t5, 0x96;\n\tlop3.b32 %3, %3, t6, t7, 0x96;\n\t}"
                                  : "+r"(l0), "+r"(l1), "+r"(l2), "+r"(l3) : "r"(a4));)
        } else if (OP == kOpLds64) {
            BSH_REP8(asm volatile("{\n\t.reg .b32 t<16>;\n\t"
                                  "ld.volatile.shared.v2.u32 {t0,t1}, [%4];\n\tld.volatile.shared.v2.u32 {t2,t3}, [%4+8192];\n\t"
                                  "ld.volatile.shared.v2.u32 {t4,t5}, [%4+16384];\n\tld.volatile.shared.v2.u32 {t6,t7}, [%4+24576];\n\t"
                                  "ld.volatile.shared.v2.u32 {t8,t9}, [%4];\n\tld.volatile.shared.v2.u32 {t10,t11}, [%4+8192];\n\t"
                                  "ld.volatile.shared.v2.u32 {t12,t13}, [%4+16384];\n\tld.volatile.shared.v2.u32 {t14,t15}, [%4+24576];\n\t"
                                  "lop3.b32 %0, %0, t0, t1, 0x96;\n\tlop3.b32 %1, %1, t2, t3, 0x96;\n\t"
                                  "lop3.b32 %2, %2, t4, t5, 0x96;\n\tlop3.b32 %3, %3, t6, t7, 0x96;\n\t"
                                  "lop3.b32 %0, %0, t8, t9, 0x96;\n\tlop3.b32 %1, %1, t10, t11, 0x96;\n\t"
                                  "lop3.b32 %2, %2, t12, t13, 0x96;\n\tlop3.b32 %3, %3, t14, t15, 0x96;\n\t}"
                                  : "+r"(l0), "+r"(l1), "+r"(l2), "+r"(l3) : "r"(a8));)
        } else {
            BSH_REP8(asm volatile("{\n\t.reg .b32 t<32>;\n\t"
                                  "ld.volatile.shared.v4.u32 {t0,t1,t2,t3}, [%4];\n\tld.volatile.shared.v4.u32 {t4,t5,t6,t7}, [%4+16384];\n\t"
                                  "ld.volatile.shared.v4.u32 {t8,t9,t10,t11}, [%4];\n\tld.volatile.shared.v4.u32 {t12,t13,t14,t15}, [%4+16384];\n\t"
                                  "ld.volatile.shared.v4.u32 {t16,t17,t18,t19}, [%4];\n\tld.volatile.shared.v4.u32 {t20,t21,t22,t23}, [%4+16384];\n\t"
                                  "ld.volatile.shared.v4.u32 {t24,t25,t26,t27}, [%4];\n\tld.volatile.shared.v4.u32 {t28,t29,t30,t31}, [%4+16384];\n\t"
                                  "lop3.b32 %0, %0, t0, t1, 0x96;\n\tlop3.b32 %1, %1, t2, t3, 0x96;\n\t"
                                  "lop3.b32 %2, %2, t4, t5, 0x96;\n\tlop3.b32 %3, %3, t6, t7, 0x96;\n\t"
                                  "lop3.b32 %0, %0, t8, t9, 0x96;\n\tlop3.b32 %1, %1, t10, t11, 0x96;\n\t"
                                  "lop3.b32 %2, %2, t12, t13, 0x96;\n\tlop3.b32 %3, %3, t14, t15, 0x96;\n\t"
                                  "lop3.b32 %0, %0, t16, t17, 0x96;\n\tlop3.b32 %1, %1, t18, t19, 0x96;\n\t"
                                  "lop3.b32 %2, %2, t20, t21, 0x96;\n\tlop3.b32 %3, %3, t22, t23, 0x96;\n\t"
                                  "lop3.b32 %0, %0, t24, t25, 0x96;\n\tlop3.b32 %1, %1, t26, t27, 0x96;\n\t"
                                  "lop3.b32 %2, %2, t28, t29, 0x96;\n\tlop3.b32 %3, %3, t30, t31, 0x96;\n\t}"
                                  : "+r"(l0), "+r"(l1), "+r"(l2), "+r"(l3) : "r"(a16));)
        }
    }
    // keep every chain alive
    const uint32_t fold = r0 ^ r1 ^ r2 ^ r3 ^ r4 ^ r5 ^ r6 ^ r7 ^ l0 ^ l1 ^ l2 ^ l3 ^
                          __float_as_uint(f0 + f1 + f2 + f3 + f4 + f5 + f6 + f7) ^
                          (uint32_t)__double2loint(d0 + d1 + d2 + d3 + d4 + d5 + d6 + d7);
    if (fold == 0x12345u) sink[0] = fold;
    __syncthreads();                                     // the block's 32 warps are done
    const long long c1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns1));
    if (threadIdx.x == 0) {
        samples[blockIdx.x].cycles = c1 - c0;
        samples[blockIdx.x].ns = ns1 - ns0;
    }
}

#undef BSH_REP8

}  // namespace bsh
