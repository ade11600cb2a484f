// mphv_probe.cuh -- issue-rate microbenchmark behind the "issue" roofline of bench.py (DESIGN.md sec. 7,
// profiles/r02_issue_rate.md): how many warp instructions per cycle one SM scheduler sustains for the
// instruction kinds the sweep kernels are made of (DFMA, DADD, 64-bit select = 2 FSEL, DSETP, IMAD), as a
// function of the warps resident per scheduler. Every thread runs ILP = 4 independent dependency chains of
// UNROLL x ops, so a single warp can keep 4 instructions in flight; time by CUDA events, cycles from the SM
// clock NVML reports during the run.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mphv {

enum { PROBE_DFMA = 0, PROBE_DADD = 1, PROBE_SEL64 = 2, PROBE_DSETP_SEL64 = 3, PROBE_IMAD = 4, PROBE_FFMA = 5,
       PROBE_MIX = 6, PROBE_DFMA3 = 7, PROBE_DADD2 = 8, PROBE_DFMA3_SEL = 9, PROBE_KINDS = 10 };
enum { PROBE_ILP = 4, PROBE_UNROLL = 16 };

// thread instructions the loop body issues per chain link, by kind (checked against cuobjdump -sass)
__host__ __device__ inline int probe_instr_per_link(int kind)
{
    switch (kind) {
    case PROBE_SEL64: return 2;          // one 64-bit select = 2 FSEL
    case PROBE_DSETP_SEL64: return 3;    // DSETP + 2 FSEL
    case PROBE_MIX: return 5;            // DADD + DSETP + 2 FSEL + DFMA: the limiter's mix
    case PROBE_DFMA3: return 3;          // three DFMA whose three operands are all live registers
    case PROBE_DADD2: return 2;          // two DADD whose two operands are both live registers
    case PROBE_DFMA3_SEL: return 3;      // one DFMA with three live operands + one 64-bit select of two live operands (2 FSEL)
    default: return 1;
    }
}

template <int KIND>
__global__ void __launch_bounds__(1024) probe_kernel(double *out, int iters, double a, double b, int ia)
{
    double x[PROBE_ILP], y[PROBE_ILP], z[PROBE_ILP];
    int n[PROBE_ILP];
    float yf[PROBE_ILP];
#pragma unroll
    for (int k = 0; k < PROBE_ILP; ++k) { x[k] = a * (threadIdx.x + k); n[k] = ia + threadIdx.x + k; yf[k] = (float)x[k]; y[k] = b * (k + 1); z[k] = a - k; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < PROBE_UNROLL; ++u) {
#pragma unroll
            for (int k = 0; k < PROBE_ILP; ++k) {
                if (KIND == PROBE_DFMA) x[k] = fma(x[k], a, b);
                else if (KIND == PROBE_DADD) x[k] = x[k] + b;
                else if (KIND == PROBE_SEL64) {
                    // predicate from the integer lane state so that no DSETP is needed; selp.f64 = 2 FSEL
                    asm volatile("{ .reg .pred p; setp.ne.s32 p, %2, 0; selp.f64 %0, %0, %1, p; }" : "+d"(x[k]) : "d"(b), "r"(n[k]));
                } else if (KIND == PROBE_DSETP_SEL64) {
                    asm volatile("{ .reg .pred p; setp.lt.f64 p, %0, %1; selp.f64 %0, %0, %2, p; }" : "+d"(x[k]) : "d"(a), "d"(b));
                } else if (KIND == PROBE_IMAD) n[k] = n[k] * ia + it;
                else if (KIND == PROBE_FFMA) yf[k] = fmaf(yf[k], (float)a, (float)b);
                else if (KIND == PROBE_DFMA3) {
                    // no operand is loop-invariant or repeated: every DFMA reads three different register pairs
                    x[k] = fma(y[k], z[k], x[k]); y[k] = fma(z[k], x[k], y[k]); z[k] = fma(x[k], y[k], z[k]);
                } else if (KIND == PROBE_DADD2) { x[k] = y[k] + x[k]; y[k] = x[k] - y[k]; }
                else if (KIND == PROBE_DFMA3_SEL) {
                    x[k] = fma(y[k], z[k], x[k]);
                    asm volatile("{ .reg .pred p; setp.ne.s32 p, %2, 0; selp.f64 %0, %0, %1, p; }" : "+d"(y[k]) : "d"(z[k]), "r"(n[k]));
                }
                else {
                    double d = x[k] + b;                                   // DADD
                    asm volatile("{ .reg .pred p; setp.lt.f64 p, %1, %0; selp.f64 %0, %1, %0, p; }" : "+d"(d) : "d"(a));   // DSETP + 2 FSEL
                    x[k] = fma(d, a, x[k]);                                // DFMA
                }
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PROBE_ILP; ++k) s += x[k] + (double)n[k] + (double)yf[k] + y[k] + z[k];
    if (s == 12345.678) out[0] = s;          // keeps the chains alive, never true in practice
}

}  // namespace mphv
