// heget-b200: run-time support shared by every generated per-process kernel file (gen_*.cu) and by the C-ABI (api.cpp).
//
// A generated file defines, for one process, the kernels of steps a3-a8 (eq. 4), a host
// launcher and a static descriptor which the library reads through heget_plugin_desc() after dlopen.  Nothing here is process specific.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "heget_dev.cuh"

namespace hg {

// ---- descriptor of one generated process (host side) -------------------------------------------------------------------
struct LaunchArgs {
    const double* d_mom;      // [n_ext][4][n_events] FP64, device
    uint64_t n_events;
    double inv_sqrt_s;        // momenta are evaluated in units of sqrt(s_hat) (reading A21)
    double out_scale;         // S * 1/4 * 1/(n_a n_b) * g^(2(n-2)) * s_hat^-(n-4)      (eqs. 4, 9, 12)
    void* d_me2;              // double[n_events] or float[n_events]
    int hel_mode;             // 0 = sum over all helicities, 1 = one Philox-drawn helicity per event, 2 = fixed configuration
    int hel_fixed;            // mode 2: index of the configuration in the kernel's own enumeration, or -1 (vanishing)
    uint64_t seed;            // mode 1
    uint64_t first_event;     // mode 1: global index of event 0 (Philox counter)
    int lanes;                // helicity lanes per event (power of two <= 32), 0 = choose
    cudaStream_t stream;
};

struct KernelInfo { int regs, local_bytes, smem_static, max_threads, block; };

struct ProcDesc {
    const char* name;           // canonical process string, e.g. "g g > g g g"
    const char* tag;
    int n_ext, n_gluons, n_quark_legs;
    int n_hel;                  // 2^n_ext, the helicity configurations of eq. 12
    int n_hel_eval;             // configurations that are not identically zero (quark-line chirality conservation)
    int n_diagrams;             // paper's convention: a four-gluon vertex counts 3 (Table 1)
    int n_topologies;
    int n_currents;             // distinct off-shell sub-currents per helicity configuration
    int n_color;                // colour basis in the paper's convention (Table 1)
    int n_color_eval;           // basis the kernel sums diagrams on
    int n_color_reduced;        // after merging elements whose J are proportional
    double sym_factor, avg_color, avg_spin;
    double flops_per_hel;       // counted from the generator's IR (per evaluated helicity configuration)
    double flops_per_event;     // prologue + n_hel_eval * flops_per_hel
    double flops_colour_per_hel;
    const double* colour_matrix;        // n_color x n_color, paper basis, without 1/(n_a n_b)  (eq. 9)
    const double* colour_matrix_eval;   // n_color_reduced x n_color_reduced
    const signed char* hel_table;       // [n_hel_eval][n_ext] physical helicities of the kernel's enumeration
    int (*launch)(int prec, const LaunchArgs&);                 // returns cudaError_t
    int (*kernel_info)(int prec, int lanes, KernelInfo*);       // registers / local memory of the compiled kernel
    int block[2];               // threads per block of the default (widest) variant, FP64 / FP32
    int lanes_wide;             // helicity lanes per event of the wide variant (power of two <= 32 dividing n_hel_eval)
    int lanes_avail;            // bit 0: the one-event-per-thread variant is compiled in, bit 1: the wide variant is
    ProcDesc* next;
    int abi_version;            // HG_ABI_VERSION of the headers the plug-in was compiled against (checked at load)
};
#define HG_ABI_VERSION 2

// every plug-in (one shared object per process) exports   extern "C" const hg::ProcDesc* heget_plugin_desc();

#if defined(HG_HOST_DEBUG)
#define HG_SMEM_DECL static unsigned char hg_smem[1 << 20]
#else
#define HG_SMEM_DECL extern __shared__ __align__(16) unsigned char hg_smem[]
#endif
#if defined(__CUDACC__) || defined(HG_HOST_DEBUG)
// ---- device helpers used by the generated code ------------------------------------------------------------------------
// Reads of the per-event cache are helicity-loop invariant: left to itself the compiler hoists all of them out of the
// helicity loop and holds ~100 values in registers for the whole body, which is what spills.  A volatile read stays where
// the schedule put it (one LDS per use, next to the vertex call that consumes it).  Measured on C2 (profiles/): FP64
// 12.6 -> 26 TFLOP/s with volatile reads (stack frame 2200 -> 730 B); FP32, whose registers hold twice as many values and
// whose FMA rate is twice as far ahead of the shared-memory pipe, is faster with the hoisted copy (56 vs 48 TFLOP/s).
template <typename T> __device__ __forceinline__ T ldc(const T* p) {
#if defined(HG_CACHE_VOLATILE32)
    constexpr bool vol = true;
#elif defined(HG_CACHE_HOISTABLE64)
    constexpr bool vol = false;
#else
    constexpr bool vol = sizeof(T) == 8;
#endif
    if constexpr (vol) return *reinterpret_cast<const volatile T*>(p); else return *p;
}
// Between two operations of the generated schedule: keeps the compiler from hoisting the next operation's cache reads (and
// with them its arithmetic) far ahead, which is what stretches live ranges beyond the schedule's own small live set.
template <typename T> __device__ __forceinline__ void fence() {
#if defined(__CUDA_ARCH__) && !defined(HG_NO_FENCE)
#if defined(HG_NO_FENCE32)
    if constexpr (sizeof(T) == 8) asm volatile("" ::: "memory");
#else
    asm volatile("" ::: "memory");
#endif
#endif
}
template <> __device__ __forceinline__ f2 ldc<f2>(const f2* p) {          // same policy as an 8-byte scalar: never hoisted
#if defined(HG_CACHE_HOISTABLE64)
    return *p;
#else
    f2 r; r.v = *reinterpret_cast<const volatile unsigned long long*>(p); return r;
#endif
}
// ---- packing of helicity configurations (1 per thread for float/double, 2 for f2) -----------------------------------
// Packed threads hold the configurations t with gluon bit `pb` cleared (first half) and set (second half).
template <typename T> struct hpack {
    static constexpr int value = 1;
    typedef T out_t;
    __device__ static __forceinline__ int expand(int t, int) { return t; }
    __device__ static __forceinline__ int index(int h, int) { return h; }
    __device__ static __forceinline__ T select(int, int) { return T(1); }
    __device__ static __forceinline__ T lam(int hidx, int j, int) { return ((hidx >> j) & 1) ? T(1) : T(-1); }
    __device__ static __forceinline__ T hsum(T v) { return v; }
};
template <> struct hpack<f2> {
    static constexpr int value = 2;
    typedef float out_t;
    __device__ static __forceinline__ int expand(int t, int pb) { return ((t >> pb) << (pb + 1)) | (t & ((1 << pb) - 1)); }
    __device__ static __forceinline__ int index(int h, int pb) { return ((h >> (pb + 1)) << pb) | (h & ((1 << pb) - 1)); }
    __device__ static __forceinline__ f2 select(int h, int pb) { return ((h >> pb) & 1) ? f2(0.f, 1.f) : f2(1.f, 0.f); }
    __device__ static __forceinline__ f2 lam(int hidx, int j, int pb) { return j == pb ? f2(-1.f, 1.f) : (((hidx >> j) & 1) ? f2(1.f) : f2(-1.f)); }
    __device__ static __forceinline__ float hsum(f2 v) { return v.lo() + v.hi(); }
};
// colour-group register accumulators for J in shared memory (emit_body.inc): 16 registers that the FP32 kernels have and the
// FP64 ones do not (measured on C4: FP32 3.2e6 -> 4.1e6 events/s, FP64 1.8e6 -> 1.3e6 with 3.5 kB of new spills)
template <typename T> __host__ __device__ constexpr bool use_groups() {
#if defined(HG_NO_GROUPS)
    return false;
#else
    return sizeof(T) == 4;
#endif
}
template <typename T> __host__ __device__ constexpr bool leaf_reload() {
#if defined(HG_LEAF_RELOAD32)
    return true;
#elif defined(HG_LEAF_HOLD64)
    return false;
#else
    return sizeof(T) == 8;
#endif
}
template <typename T> __device__ __forceinline__ mom4<T> ldk(const T* ev, int slot, int stride) {
    mom4<T> k;
    k.p[0] = ldc(ev + (slot + 0) * stride); k.p[1] = ldc(ev + (slot + 1) * stride); k.p[2] = ldc(ev + (slot + 2) * stride); k.p[3] = ldc(ev + (slot + 3) * stride);
    return k;
}
template <typename T> __device__ __forceinline__ vec4<T> ldv(const T* ev, int slot, int stride, T lambda) {   // vxxxxx, helicity part
    vec4<T> w;
    w.v[0] = mk<T>(T(0), T(0));
    w.v[1] = mk<T>(lambda * ldc(ev + (slot + 0) * stride), ldc(ev + (slot + 3) * stride));
    w.v[2] = mk<T>(lambda * ldc(ev + (slot + 1) * stride), ldc(ev + (slot + 4) * stride));
    w.v[3] = mk<T>(lambda * ldc(ev + (slot + 2) * stride), ldc(ev + (slot + 5) * stride));
    return w;
}
template <typename T> __device__ __forceinline__ sp2<T> ldi(const T* ev, int slot, int stride, T chi) {       // ixxxxx, helicity part
    const T s[3] = {ldc(ev + slot * stride), ldc(ev + (slot + 1) * stride), ldc(ev + (slot + 2) * stride)};
    return ixxxxx<T>(s, chi);
}
template <typename T> __device__ __forceinline__ sp2<T> ldo(const T* ev, int slot, int stride, T chi) {       // oxxxxx, helicity part
    const T s[3] = {ldc(ev + slot * stride), ldc(ev + (slot + 1) * stride), ldc(ev + (slot + 2) * stride)};
    return oxxxxx<T>(s, chi);
}

// Philox4x32-10 (Salmon et al., SC'11): the counter-based generator of steps a1 and of HEL_SAMPLE (reading A17)
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t* out) {
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
#endif

}  // namespace hg
