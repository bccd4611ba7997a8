// FP64 peak probe (nbs_probe_fp64, include/nbs.h): register-resident instruction mixes on every SM, timed with
// CUDA events.  bench.py runs it in the same process and under the same clock sampler as the timed steps; the
// DMMA-only figure is the denominator of `roofline.frac` for the product kernel.
//   mode 0: DMMA.8x8x4 only            mode 1: DFMA only            mode 2: DADD only
//   mode 3: 12 DMMA + 12 DADD  (one k-step of the 16x16 accumulator class of k_product: 8 gather subtractions,
//           4 Gauss sums, 12 MMAs)
//   mode 4: 16 DMMA + 24 DADD  (one k-step of the 64x4 class)
#pragma once
#include <cuda_runtime.h>

#include "nbs_product.cuh"
#include "nbs_product_c.cuh"

namespace nbs {

constexpr int PROBE_THREADS = 512; // 16 warps per CTA, one CTA per SM: 4 warps per SM sub-partition
//   mode 5: 12 DADD, then 12 DMMA, order pinned (volatile asm)    mode 6: DADD and DMMA strictly alternating, order pinned
//   mode 7 / 8: mode 6 with 8 / 4 independent integer instructions per DADD + DMMA pair
__host__ __device__ constexpr int probe_dmma(int mode) { return mode == 0 ? 16 : mode == 3 ? 12 : mode == 4 ? 16 : mode >= 5 ? 12 : 0; }
__host__ __device__ constexpr int probe_dfma(int mode) { return mode == 1 ? 16 : 0; }
__host__ __device__ constexpr int probe_dadd(int mode) { return mode == 2 ? 16 : mode == 3 ? 12 : mode == 4 ? 24 : mode >= 5 ? 12 : 0; }
__device__ __forceinline__ void dmma884_v(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void dadd_v(double& d, double a, double b) {
    asm volatile("add.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b));
}

template <int MODE>
__global__ void __launch_bounds__(PROBE_THREADS, 1) k_probe_fp64(int iters, double delta, double* __restrict__ sink) {
    const int lane = threadIdx.x & 31;
    double acc[16][2];
#pragma unroll
    for (int i = 0; i < 16; ++i) { acc[i][0] = 0.0; acc[i][1] = 0.0; }
    double v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = 1.0 + 1e-3 * (lane + i);
    double w[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = 0.5 + 1e-3 * (lane - i);
    unsigned iw[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) iw[i] = lane + i;
    for (int it = 0; it < iters; ++it) {
        if (MODE == 0) {
#pragma unroll
            for (int i = 0; i < 16; ++i) dmma884(acc[i][0], acc[i][1], v[i & 7], v[8 + (i & 7)]);
        } else if (MODE == 1) {
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[i][0] = fma(v[i], delta, acc[i][0]);
        } else if (MODE == 2) {
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[i][0] += delta;
        } else if (MODE == 3) {
            // A[2], B[2] complex: 8 subtractions (eq. 4.2 gathers), 4 Gauss sums, 12 MMAs (mma_square)
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = v[i] - delta;
            const double sA0 = v[0] + v[1], sA1 = v[2] + v[3], sB0 = v[4] + v[5], sB1 = v[6] + v[7];
            const double Ar[2] = {v[0], v[2]}, Ai[2] = {v[1], v[3]}, Br[2] = {v[4], v[6]}, Bi[2] = {v[5], v[7]};
            const double sA[2] = {sA0, sA1}, sB[2] = {sB0, sB1};
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    dmma884(acc[(i * 2 + j) * 3 + 0][0], acc[(i * 2 + j) * 3 + 0][1], Ar[i], Br[j]);
                    dmma884(acc[(i * 2 + j) * 3 + 1][0], acc[(i * 2 + j) * 3 + 1][1], Ai[i], Bi[j]);
                    dmma884(acc[(i * 2 + j) * 3 + 2][0], acc[(i * 2 + j) * 3 + 2][1], sA[i], sB[j]);
                }
        } else if (MODE == 5) {
#pragma unroll
            for (int i = 0; i < 12; ++i) dadd_v(v[i], v[i], delta);
#pragma unroll
            for (int i = 0; i < 12; ++i) dmma884_v(acc[i][0], acc[i][1], v[i], v[(i + 1) % 12]);
        } else if (MODE == 7 || MODE == 8) {
            // mode 5 plus integer work between the FP64 instructions (order pinned): 4 (mode 7) or 2 (mode 8) per FP64 op
#pragma unroll
            for (int i = 0; i < 12; ++i) {
                dadd_v(v[i], v[i], delta);
#pragma unroll
                for (int k = 0; k < (MODE == 7 ? 4 : 2); ++k) asm volatile("xor.b32 %0, %0, %1;" : "+r"(iw[(i + k) & 7]) : "r"(it));
                dmma884_v(acc[i][0], acc[i][1], v[(i + 4) % 12], v[(i + 5) % 12]);
#pragma unroll
                for (int k = 0; k < (MODE == 7 ? 4 : 2); ++k) asm volatile("xor.b32 %0, %0, %1;" : "+r"(iw[(i + k + 4) & 7]) : "r"(it));
            }
        } else if (MODE == 6) {
#pragma unroll
            for (int i = 0; i < 12; ++i) {
                dadd_v(v[i], v[i], delta);
                dmma884_v(acc[i][0], acc[i][1], v[(i + 4) % 12], v[(i + 5) % 12]);
            }
        } else {
            // A[4][2] complex (16 subtractions), B entry (8 adds), 16 MMAs (mma_wide)
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = v[i] - delta;
#pragma unroll
            for (int i = 0; i < 4; ++i) w[i] = w[i] + delta;
            const double b1 = (w[0] + w[1]) + w[4], b2 = (w[2] + w[3]) + w[5]; // 4 + 4 adds: the 8-term B entry
#pragma unroll
            for (int i = 0; i < 8; ++i) dmma884(acc[i][0], acc[i][1], v[2 * i], b1);
#pragma unroll
            for (int i = 0; i < 8; ++i) dmma884(acc[i][0], acc[i][1], v[2 * i + 1], b2);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += acc[i][0] + acc[i][1];
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i];
#pragma unroll
    for (int i = 0; i < 8; ++i) s += (double)iw[i];
    if (s == 1.2345e-300) sink[blockIdx.x * PROBE_THREADS + threadIdx.x] = s; // keeps the arithmetic alive
}

// k-step probe (nbs_probe_kstep, include/nbs.h): the unit code of k_product_c in isolation.  Every one of `ncw`
// warps per CTA (one CTA per SM) runs the SAME device functions the kernel runs -- run_unit_square_c (cls 0) or
// run_unit_wide_c (cls 2) -- `reps` times on a synthetic unit of one diagram with `nsteps` k-steps: two compact blocks
// in shared memory, packed gather words from L2 with bank-conflict-free offsets (the residue rule of
// nbs_tables.hpp), another table region every repetition.  cyc[CTA * 12 + warp] = cycles of the warp's loop.
constexpr int PROBE_KSTEP_THREADS = 384; // up to 12 warps per SM, 168 registers: no setmaxnreg needed
__global__ void __launch_bounds__(PROBE_KSTEP_THREADS, 1) k_probe_kstep(const uint32_t* __restrict__ tab, int cls, int nsteps, int reps,
                                                              int ncw, double2* __restrict__ out, long long* __restrict__ cyc) {
    extern __shared__ __align__(128) char prod_smem[];
    char* sm = prod_smem;
    __shared__ int item[12];
    __shared__ __align__(16) Diag3Rec drec[PROBE_KSTEP_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (uint32_t i = tid; i < C_BLOCKS_BYTES / 16; i += blockDim.x)
        reinterpret_cast<double2*>(sm)[i] = make_double2(1e-3 * (double)(i % 97), -2e-3 * (double)(i % 89));
    if (tid == 0) { // B~1 in slot 0, B~2 in slot 1, both compact
        item[5] = (int)c_slot_base(0); item[6] = (int)c_slot_base(1);
        item[7] = item[8] = AS_PLANE * 16;
    }
    __syncthreads();
    if (warp >= ncw) return;
    Unit3Rec u;
    u.diag_begin = warp; u.diag_end = warp + 1; u.cls = cls; u.slot = 0;
    double2* o = out + ((size_t)blockIdx.x * (PROBE_KSTEP_THREADS / 32) + warp) * 256;
    const long long t0 = clock64();
    for (int r = 0; r < reps; ++r) {
        if (lane == 0) {
            Diag3Rec d;
            d.offA = (uint32_t)(((r * (PROBE_KSTEP_THREADS / 32) + warp) % 16) * 4096); d.offB = 65536u + d.offA;
            d.sbeg = 0; d.send = (uint16_t)nsteps; d.nwA = 1; d.nwB = (uint8_t)(cls >= 2 ? 4 : 1); d.K = (uint16_t)(4 * nsteps);
            drec[warp] = d;
        }
        __syncwarp();
#ifdef NBS_PROF
        long long pf[PF_N] = {};
        if (cls < 2) run_unit_square_c(u, drec, tab, sm, item, o, lane, pf);
#else
        if (cls < 2) run_unit_square_c(u, drec, tab, sm, item, o, lane);
#endif
        else run_unit_wide_c(u, drec, tab, sm, item, o, lane);
        __syncwarp();
    }
    if (lane == 0) cyc[blockIdx.x * (PROBE_KSTEP_THREADS / 32) + warp] = clock64() - t0;
}
constexpr int PROBE_KSTEP_MAX_STEPS = 48;        // a table region holds 4096 words = 64 k-steps of the widest table
constexpr size_t PROBE_KSTEP_TAB_WORDS = 1 << 17; // A tables in the first half, B tables in the second

} // namespace nbs
