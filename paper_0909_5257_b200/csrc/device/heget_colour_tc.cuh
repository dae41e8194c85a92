// heget-b200: the colour stage as a batched tensor-core contraction (step a7 for large colour bases; SURVEY.md 8(a) "a7-TC").
//
// PAPER.md:91 (eq. 10): sum_ab J_a^* C_ab J_b = Jr^T C Jr + Ji^T C Ji -- for many (event, helicity configuration) pairs at once
// this is Y = X C with X = [rows x R], one row per (event, configuration, re/im), followed by the row-wise product sum_a X_a Y_a
// (with 120 colour elements the paper's time went into exactly this step).
// The table kernel (heget_tab.cuh, colour stage 3) writes the rows of X to HBM instead of contracting them itself; this kernel
// contracts them on the tensor cores:
//   FP32: mma.sync m16n8k8 TF32 with a 3-term error-compensated split, x = hi + lo (hi = tf32(x), lo = tf32(x - hi)) on both
//         operands: X C ~ Xhi Chi + Xhi Clo + Xlo Chi, FP32 accumulators -- relative error ~2^-21 instead of TF32's 2^-11;
//   FP64: mma.sync m8n8k4 DMMA (tcgen05 has no f64 kind).
// C (symmetric, padded to a multiple of 8) sits in shared memory, split into hi / lo for TF32; every warp owns 16 (8 in FP64)
// rows of X, reads its A fragments straight from global memory (each element once) and keeps the whole row block of Y in
// accumulators; the epilogue multiplies by X again and reduces over the colour index inside the quad.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace hg {

#if defined(__CUDACC__)
__device__ __forceinline__ unsigned tf32_of(float x) { unsigned r; asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x)); return r; }
__device__ __forceinline__ void mma_tf32(float* c, const unsigned* a, unsigned b0, unsigned b1) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma_f64(double* c, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// X: [n_rows][Rp] row-major (Rp = padded colour dimension, a multiple of 8, <= 128); Cm: [Rp][Rp] symmetric; form[row] = sum_ab X_a C_ab X_b
constexpr int TC_MAX_NT = 16;      // n-tiles of 8 columns: Rp <= 128

__global__ void __launch_bounds__(256) k_colour_tf32(const float* __restrict__ X, const float* __restrict__ Cm, float* __restrict__ form, const unsigned long long n_rows, const int Rp) {
    extern __shared__ __align__(16) unsigned char tc_smem[];
    const int pitch = Rp + 8;                          // pitch = 8 mod 32 words: the B-fragment reads (k = lane % 4, n = lane / 4) hit 32 different banks
    unsigned* chi = reinterpret_cast<unsigned*>(tc_smem);
    unsigned* clo = chi + (size_t)Rp * pitch;
    for (int i = threadIdx.x; i < Rp * Rp; i += blockDim.x) {
        const int r = i / Rp, c = i % Rp;
        const float v = Cm[i];
        const unsigned h = tf32_of(v);
        chi[r * pitch + c] = h; clo[r * pitch + c] = tf32_of(v - __uint_as_float(h));
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3, nt = Rp / 8;
    const unsigned long long r0 = ((unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 16;
    if (r0 >= n_rows) return;
    const unsigned long long ra = min(r0 + g, n_rows - 1), rb = min(r0 + g + 8, n_rows - 1);
    const float* xa = X + ra * Rp; const float* xb = X + rb * Rp;
    float acc[TC_MAX_NT][4];
#pragma unroll
    for (int j = 0; j < TC_MAX_NT; ++j) { acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.f; }
    for (int kt = 0; kt < nt; ++kt) {
        const float av[4] = {xa[kt * 8 + t], xb[kt * 8 + t], xa[kt * 8 + t + 4], xb[kt * 8 + t + 4]};
        unsigned ah[4], al[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { ah[i] = tf32_of(av[i]); al[i] = tf32_of(av[i] - __uint_as_float(ah[i])); }
        const unsigned* bh = chi + (kt * 8 + t) * pitch + g;
        const unsigned* bl = clo + (kt * 8 + t) * pitch + g;
#pragma unroll
        for (int j = 0; j < TC_MAX_NT; ++j) if (j < nt) {
            const unsigned h0 = bh[j * 8], h1 = bh[4 * pitch + j * 8], l0 = bl[j * 8], l1 = bl[4 * pitch + j * 8];
            mma_tf32(acc[j], al, h0, h1);        // small terms first
            mma_tf32(acc[j], ah, l0, l1);
            mma_tf32(acc[j], ah, h0, h1);
        }
    }
    // row-wise product with X: thread holds Y[row g][2t, 2t+1] and Y[row g+8][2t, 2t+1] of every n-tile
    float fa = 0.f, fb = 0.f;
#pragma unroll
    for (int j = 0; j < TC_MAX_NT; ++j) if (j < nt) {
        const float2 va = *reinterpret_cast<const float2*>(xa + j * 8 + 2 * t), vb = *reinterpret_cast<const float2*>(xb + j * 8 + 2 * t);
        fa += acc[j][0] * va.x + acc[j][1] * va.y; fb += acc[j][2] * vb.x + acc[j][3] * vb.y;
    }
    fa += __shfl_xor_sync(0xffffffffu, fa, 1); fa += __shfl_xor_sync(0xffffffffu, fa, 2);
    fb += __shfl_xor_sync(0xffffffffu, fb, 1); fb += __shfl_xor_sync(0xffffffffu, fb, 2);
    if (t == 0) { if (r0 + g < n_rows) form[r0 + g] = fa; if (r0 + g + 8 < n_rows) form[r0 + g + 8] = fb; }
}

__global__ void __launch_bounds__(256) k_colour_dmma(const double* __restrict__ X, const double* __restrict__ Cm, double* __restrict__ form, const unsigned long long n_rows, const int Rp) {
    extern __shared__ __align__(16) unsigned char tc_smem[];
    const int pitch = Rp + 4;                          // pitch = 4 mod 16 doubles: the B-fragment reads (k = lane % 4, n = lane / 4) are conflict free
    double* cs = reinterpret_cast<double*>(tc_smem);
    for (int i = threadIdx.x; i < Rp * Rp; i += blockDim.x) cs[(i / Rp) * pitch + (i % Rp)] = Cm[i];
    __syncthreads();
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3, nt = Rp / 8;
    const unsigned long long r0 = ((unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 8;
    if (r0 >= n_rows) return;
    const unsigned long long ra = min(r0 + g, n_rows - 1);
    const double* xa = X + ra * Rp;
    double acc[TC_MAX_NT][2];
#pragma unroll
    for (int j = 0; j < TC_MAX_NT; ++j) { acc[j][0] = acc[j][1] = 0.0; }
    for (int kt = 0; kt < Rp / 4; ++kt) {
        const double a = xa[kt * 4 + t];
        const double* b = cs + (kt * 4 + t) * pitch + g;
#pragma unroll
        for (int j = 0; j < TC_MAX_NT; ++j) if (j < nt) mma_f64(acc[j], a, b[j * 8]);
    }
    double f = 0.0;
#pragma unroll
    for (int j = 0; j < TC_MAX_NT; ++j) if (j < nt) { const double2 v = *reinterpret_cast<const double2*>(xa + j * 8 + 2 * t); f += acc[j][0] * v.x + acc[j][1] * v.y; }
    f += __shfl_xor_sync(0xffffffffu, f, 1); f += __shfl_xor_sync(0xffffffffu, f, 2);
    if (t == 0 && r0 + g < n_rows) form[r0 + g] = f;
}

// helicity sum (eq. 12): me2[e] = scale * sum over the rows of event e (configurations x re/im; rows of padding lanes hold zeros)
template <typename T>
__global__ void k_colour_finish(const T* __restrict__ form, T* __restrict__ me2, const unsigned long long n_events, const int rows_per_event, const double scale) {
    const unsigned long long e = (unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (e >= n_events) return;
    const int lane = threadIdx.x & 31;
    T s = T(0);
    for (int r = lane; r < rows_per_event; r += 32) s += form[e * rows_per_event + r];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) me2[e] = (T)(scale * (double)s);
}
#endif

}  // namespace hg
