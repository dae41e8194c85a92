// heget-b200: the TABLE-DRIVEN evaluator of steps a3-a8 (eq. 4) -- one generic kernel per
// precision that interprets the table program the generator (csrc/gen/tab.hpp) writes for a process.  No per-process code:
// the whole kernel is a few kB of instructions, so the instruction cache holds it (the straight-line kernels of the big
// processes were instruction-fetch bound).
//
// Work decomposition (one CTA = EPC slots x WPE chunks of 32 configurations x NSP warps; a slot is one event, or two for the packed type):
//   prologue  once per event, FP64: momenta in units of sqrt(s_hat) staged in shared memory; the momentum of every leg subset
//             that carries a current and its 1/q^2; the external wavefunctions ixxxxx/oxxxxx/vxxxxx of both helicities
//              written to the event's current store.
//   phase A   off-shell currents jvvxx0 / jgggx0 / jioxx0 / fvixx0 / fvoxx0, level by level
//             (2-leg, 3-leg, ...).  A lane owns one (current, helicity variant) pair: a current over the leg set S is
//             evaluated once per 2^|S| helicity assignment of ITS legs and kept in shared memory for the whole event
//             (helicity recycling, SURVEY.md 8(d) "factorised").  A merged current is the sum of several vertex terms.
//   phase B   a warp owns 32 helicity configurations of the event (lane = configuration) and walks the closing list:
//             amplitude = vvvxxx / ggggxx / iovxx0 of three or four stored currents, the variant of each
//             picked by the lane's helicity bits; amplitudes of one colour group are summed in a register, then
//             J_k += x_gk S_g (eq. 8) on the lane's column of J in shared memory.
//   phase C   colour form  Jr^T C Jr + Ji^T C Ji (eq. 10) per lane, register-tiled over 8 rows, C streamed through
//             the warp's ring by cp.async; helicity sum (eq. 12) by warp shuffles; me2 = out_scale * sum.
// Several warps per block of J (NSP > 1, chosen by api.cu for the processes whose J fills the tensor memory with four warps): the
// colour groups are dealt out to the NSP warps two at a time; every warp evaluates the closings of its groups and parks the finished
// group sums S_g in a FIFO of its own in shared memory, and applies J_k += x_gk S_g itself when its TURN comes: the turn goes round
// the warps in the order in which the groups were dealt (an mbarrier per warp, one phase per turn), so the additions into every J_k
// happen in the ORIGINAL group order and |M|^2 is bit-identical for every NSP (tests/test_gpu_parity.py).  All NSP warps share
// phase A and split the row tiles of phase C.
// Current store layout: 16-byte chunks; a current with nv variants and ncomp complex components occupies
// chunk(q, v) = base + q * nv + v, each chunk holding 2 complex (FP32) or 1 complex (FP64) -- lanes that share a variant read
// the same chunk (multicast), lanes with different variants read neighbouring chunks (no bank conflict).
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#include "heget_dev.cuh"
#include "heget_rt.cuh"

namespace hg {

struct TabDev {
    int n_ext, NH, nchunks, cpc, R, Rpad, nK, store32, n_levels, n_closings;
    const uint32_t* kmask; const uint32_t* leginfo;
    const uint32_t* a_hdr; const uint32_t* a_out; const uint32_t* a_term; const uint32_t* a_level;
    int n_entries, n_rows;
    const unsigned char* b_ent;  // [n_entries + padding] closing records in the byte layout of this precision (tab_entry_bytes<T>() each; api.cu, table_to_device)
    const unsigned char* lanerows; // [n_rows][nchunks * 32] per-lane bytes: variant of a leg set, or validity | chirality << 1
    const void* coef;            // T[]: pool of rational coefficients
    const void* cmat;            // T[(Rpad/8 + 1) * Rpad * 8]: tiles of the colour matrix (cstage 0), of its Cholesky factor (cstage 2)
    int cstage;                  // colour stage: 0 symmetric form with literal coefficients, 1 distinct-value table + index map (the paper's scheme), 2 Cholesky factor |L^T J|^2, 3 J handed to the tensor-core kernel
    void* jout;                  // cstage 3: rows of J written to HBM for the tensor-core contraction (heget_colour_tc.cuh): out_t[(event * nchunks * 32 + configuration) * 2 + re/im][Rpad]
    const unsigned char* cidx;   // cstage 1: index of every coefficient of cmat in cvals
    const void* cvals;           // cstage 1: T[<= 256] distinct coefficient values
    const short* evalidx;        // [2^n_ext] helicity bits -> evaluated configuration or -1
    // nsp > 1: nsp warps serve one (slot, chunk).  Warp s walks list s of the closing records (the colour groups dealt out gpt at a time,
    // in turn), keeps finished group sums in its FIFO and applies them to J when its turn comes -- turn k of warp s after turn k of warp
    // s - 1 (turn k - 1 of the last warp for s = 0): the original group order, so J and |M|^2 are bit-identical to the one-warp walk.
    int nsp, gpt;
    int list0[4], nrec[4], ngrp[4];   // list s: first record (index into b_ent), records, colour groups
};

// shared-memory bytes of one event (momenta slots + store) and of one warp's J column block
template <typename T> __host__ __device__ inline size_t tab_event_bytes(int nK, int store32) {
    return (size_t)nK * 4 * sizeof(T) + (((size_t)nK * sizeof(T) + 15) / 16) * 16 + (size_t)store32 * 16 * (sizeof(T) / 4);
}
template <typename T> __host__ __device__ inline size_t tab_warp_bytes(int R) { return (size_t)2 * R * 32 * sizeof(T); }
// a closing record is 96 bytes for float (8 header words + 8 colour updates of 8 bytes) and 192 bytes for the 8-byte element types
// (12 header words + 8 updates of 16 bytes); every warp keeps a ring of TAB_RING of them in shared memory.
// After phase B the ring double-buffers the blocks of the colour matrix (64 coefficients = 256 / 512 bytes each).
template <typename T> __host__ __device__ constexpr int tab_entry_bytes() { return sizeof(T) == 4 ? 96 : 192; }
#define HG_TAB_RING 16
#define HG_TAB_MAXU 8
#ifndef HG_TAB_QD
#define HG_TAB_QD 4
#endif
// one FIFO entry (a finished group sum waiting for its warp's turn): S_g of the 32 lanes, a header word (updates | last-of-group << 8) in a 16-byte line, the 8 updates of the record
template <typename T> __host__ __device__ constexpr int tab_queue_bytes() { return 32 * 2 * (int)sizeof(T) + 16 + HG_TAB_MAXU * (sizeof(T) == 4 ? 8 : 16); }
// per warp: its turn mbarrier (32 arrivals per phase: every lane, when a turn of the warp is complete) in a 16-byte line + the FIFO entries
#define HG_TAB_QHDR 16
template <typename T> __host__ __device__ constexpr int tab_qblock_bytes() { return HG_TAB_QHDR + HG_TAB_QD * tab_queue_bytes<T>(); }
template <typename T> __host__ __device__ inline size_t tab_rows_bytes(int n_rows, int nchunks) { return (((size_t)n_rows * nchunks * 32) + 15) / 16 * 16; }
template <typename T> inline size_t tab_smem_bytes(const TabDev& d, int epc, bool j_in_tmem = false, int nsp = 1) {
    const int ev = sizeof(T) == 8 && !std::is_same<T, double>::value ? 2 : 1;      // events per slot
    return (size_t)epc * (sizeof(double) * 4 * d.n_ext * ev + tab_event_bytes<T>(d.nK, d.store32)
                          + (size_t)d.nchunks * ((j_in_tmem ? 0 : tab_warp_bytes<T>(d.R)) + (size_t)nsp * HG_TAB_RING * tab_entry_bytes<T>() + (nsp > 1 ? (size_t)nsp * tab_qblock_bytes<T>() : 0))
                          + sizeof(double) * d.nchunks * 3 * ev)
           + tab_rows_bytes<T>(d.n_rows, d.nchunks);
}

#if defined(__CUDACC__)
#ifdef HG_TAB_TIMING
__device__ unsigned long long g_tab_timing[16];
#endif
// ---- element traits ------------------------------------------------------------------------------------------------------------
// T = double: FP64.  T = float: FP32, one event per warp.  T = f2 (heget_dev.cuh): FP32 on packed f32x2 instructions (FFMA2 / FMUL2 /
// FADD2), the two halves being TWO EVENTS that walk the table together: every arithmetic instruction, every table word, every address
// computation serves both, which halves the issue slots per event of a kernel that is issue-bound in FP32.
template <typename T> struct el;
template <> struct el<float> {
    static constexpr int EV = 1; typedef float out_t;
    static __device__ __forceinline__ float pack(double a, double) { return (float)a; }
    static __device__ __forceinline__ float half(float v, int) { return v; }
};
template <> struct el<double> {
    static constexpr int EV = 1; typedef double out_t;
    typedef double2 v2;                    // one 16-byte chunk = (re, im), loaded as a native vector: no register shuffling
    static __device__ __forceinline__ double get(double x) { return x; }
    static __device__ __forceinline__ double put(double x) { return x; }
    static __device__ __forceinline__ double pack(double a, double) { return a; }
    static __device__ __forceinline__ double half(double v, int) { return v; }
    static __device__ __forceinline__ double from_bits(unsigned lo, unsigned hi) { return __hiloint2double((int)hi, (int)lo); }
    static __device__ __forceinline__ unsigned lo(double v) { return (unsigned)__double2loint(v); }
    static __device__ __forceinline__ unsigned hi(double v) { return (unsigned)__double2hiint(v); }
};
template <> struct el<f2> {
    static constexpr int EV = 2; typedef float out_t;
    typedef ulonglong2 v2;
    static __device__ __forceinline__ f2 get(unsigned long long x) { f2 r; r.v = x; return r; }
    static __device__ __forceinline__ unsigned long long put(f2 x) { return x.v; }
    static __device__ __forceinline__ f2 pack(double a, double b) { return f2((float)a, (float)b); }
    static __device__ __forceinline__ float half(f2 v, int j) { return j ? v.hi() : v.lo(); }
    static __device__ __forceinline__ f2 from_bits(unsigned lo, unsigned hi) { f2 r; r.v = ((unsigned long long)hi << 32) | lo; return r; }
    static __device__ __forceinline__ unsigned lo(f2 v) { return (unsigned)v.v; }
    static __device__ __forceinline__ unsigned hi(f2 v) { return (unsigned)(v.v >> 32); }
};
template <typename T> __device__ __forceinline__ cx<T> cx_ld(const void* p) { const typename el<T>::v2 u = *reinterpret_cast<const typename el<T>::v2*>(p); return mk<T>(el<T>::get(u.x), el<T>::get(u.y)); }
template <typename T> __device__ __forceinline__ void cx_st(void* p, const cx<T>& c) { typename el<T>::v2 u; u.x = el<T>::put(c.re); u.y = el<T>::put(c.im); *reinterpret_cast<typename el<T>::v2*>(p) = u; }

template <typename T> struct tabio {       // 8-byte elements (double, f2): one complex per 16-byte chunk
    // chunk of (current base32 b, variant v): 2 b + q nv + v; addr = b + v with b a multiple of nv
    static __device__ __forceinline__ unsigned a64(unsigned addr, unsigned lnv) { const unsigned m = (1u << lnv) - 1u; return 2u * (addr & ~m) + (addr & m); }
    static __device__ __forceinline__ vec4<T> ldv(const unsigned char* st, unsigned addr, unsigned lnv) {
        const uint4* s = reinterpret_cast<const uint4*>(st) + a64(addr, lnv);
        const unsigned nv = 1u << lnv;
        vec4<T> w; w.v[0] = cx_ld<T>(s); w.v[1] = cx_ld<T>(s + nv); w.v[2] = cx_ld<T>(s + 2 * nv); w.v[3] = cx_ld<T>(s + 3 * nv); return w;
    }
    static __device__ __forceinline__ void stv(unsigned char* st, unsigned addr, unsigned lnv, const vec4<T>& w) {
        uint4* s = reinterpret_cast<uint4*>(st) + a64(addr, lnv);
        const unsigned nv = 1u << lnv;
        cx_st<T>(s, w.v[0]); cx_st<T>(s + nv, w.v[1]); cx_st<T>(s + 2 * nv, w.v[2]); cx_st<T>(s + 3 * nv, w.v[3]);
    }
    static __device__ __forceinline__ sp2<T> lds(const unsigned char* st, unsigned addr, unsigned lnv) {
        const uint4* s = reinterpret_cast<const uint4*>(st) + a64(addr, lnv);
        sp2<T> f; f.s[0] = cx_ld<T>(s); f.s[1] = cx_ld<T>(s + (1u << lnv)); return f;
    }
    static __device__ __forceinline__ void sts(unsigned char* st, unsigned addr, unsigned lnv, const sp2<T>& f) {
        uint4* s = reinterpret_cast<uint4*>(st) + a64(addr, lnv);
        cx_st<T>(s, f.s[0]); cx_st<T>(s + (1u << lnv), f.s[1]);
    }
    static __device__ __forceinline__ mom4<T> ldk(const T* evk, unsigned slot) {
        const uint4* s = reinterpret_cast<const uint4*>(evk) + 2 * slot;
        const cx<T> a = cx_ld<T>(s), b = cx_ld<T>(s + 1);
        mom4<T> k; k.p[0] = a.re; k.p[1] = a.im; k.p[2] = b.re; k.p[3] = b.im; return k;
    }
};
template <> struct tabio<float> {
    static __device__ __forceinline__ vec4<float> ldv(const unsigned char* st, unsigned addr, unsigned lnv) {
        const float4* s = reinterpret_cast<const float4*>(st);
        const float4 c0 = s[addr], c1 = s[addr + (1u << lnv)];
        vec4<float> w; w.v[0] = mk<float>(c0.x, c0.y); w.v[1] = mk<float>(c0.z, c0.w); w.v[2] = mk<float>(c1.x, c1.y); w.v[3] = mk<float>(c1.z, c1.w); return w;
    }
    static __device__ __forceinline__ void stv(unsigned char* st, unsigned addr, unsigned lnv, const vec4<float>& w) {
        float4* s = reinterpret_cast<float4*>(st);
        s[addr] = make_float4(w.v[0].re, w.v[0].im, w.v[1].re, w.v[1].im); s[addr + (1u << lnv)] = make_float4(w.v[2].re, w.v[2].im, w.v[3].re, w.v[3].im);
    }
    static __device__ __forceinline__ sp2<float> lds(const unsigned char* st, unsigned addr, unsigned) {
        const float4 c = reinterpret_cast<const float4*>(st)[addr];
        sp2<float> f; f.s[0] = mk<float>(c.x, c.y); f.s[1] = mk<float>(c.z, c.w); return f;
    }
    static __device__ __forceinline__ void sts(unsigned char* st, unsigned addr, unsigned, const sp2<float>& f) {
        reinterpret_cast<float4*>(st)[addr] = make_float4(f.s[0].re, f.s[0].im, f.s[1].re, f.s[1].im);
    }
    static __device__ __forceinline__ mom4<float> ldk(const float* evk, unsigned slot) {
        const float4 c = reinterpret_cast<const float4*>(evk)[slot];
        mom4<float> k; k.p[0] = c.x; k.p[1] = c.y; k.p[2] = c.z; k.p[3] = c.w; return k;
    }
};

template <typename T> __device__ __forceinline__ void vacc(vec4<T>& a, const vec4<T>& b) {
#pragma unroll
    for (int m = 0; m < 4; ++m) { a.v[m].re += b.v[m].re; a.v[m].im += b.v[m].im; }
}
template <typename T> __device__ __forceinline__ void sacc(sp2<T>& a, const sp2<T>& b) {
    a.s[0].re += b.s[0].re; a.s[0].im += b.s[0].im; a.s[1].re += b.s[1].re; a.s[1].im += b.s[1].im;
}


// ---- phase B helpers ------------------------------------------------------------------------------------------------------
// operands of one closing in registers: VVV w[0..3] = a, w[4..7] = b, w[8..11] = c, k = (ka, kb, kc); GGGG w[0..15] = a, b, c, d;
// IOV w[0..1] = psi, w[2..3] = psibar, w[4..7] = gluon
template <typename T> struct TabOps { cx<T> w[16]; T k[12]; };

template <typename T> __device__ __forceinline__ void tab_ld(cx<T>* w, const unsigned char* store, unsigned addr, unsigned stride, int ncomp) {      // 8-byte elements
    const uint4* s = reinterpret_cast<const uint4*>(store) + addr;
    w[0] = cx_ld<T>(s); w[1] = cx_ld<T>(s + stride);
    if (ncomp == 4) { w[2] = cx_ld<T>(s + 2 * stride); w[3] = cx_ld<T>(s + 3 * stride); }
}
template <> __device__ __forceinline__ void tab_ld<float>(cx<float>* w, const unsigned char* store, unsigned addr, unsigned stride, int ncomp) {
    const float4* s = reinterpret_cast<const float4*>(store) + addr;
    const float4 c0 = s[0]; w[0] = mk<float>(c0.x, c0.y); w[1] = mk<float>(c0.z, c0.w);
    if (ncomp == 4) { const float4 c1 = s[stride]; w[2] = mk<float>(c1.x, c1.y); w[3] = mk<float>(c1.z, c1.w); }
}
template <typename T> __device__ __forceinline__ void tab_ldk4(T* k, const T* p) {      // 8-byte elements
    const cx<T> a = cx_ld<T>(p), b = cx_ld<T>(reinterpret_cast<const uint4*>(p) + 1);
    k[0] = a.re; k[1] = a.im; k[2] = b.re; k[3] = b.im;
}
template <> __device__ __forceinline__ void tab_ldk4<float>(float* k, const float* p) { const float4 c = *reinterpret_cast<const float4*>(p); k[0] = c.x; k[1] = c.y; k[2] = c.z; k[3] = c.w; }
// closing record (uniform, in the warp's ring).  Word 0: kind (0 vvv, 1 gggg, 2 iov, 3 updates only) | reset S << 2 | updates << 3 |
// byte offset of the flag row << 16; words 1-2: chunk bases of the operands a | b << 16, c | d << 16; words 3-4: byte offsets of their
// variant rows; word 5: strides (chunks between the 16-byte pieces of one variant) a | b << 8 | c << 16 | d << 24; word 6: byte offsets
// of K_a | K_b << 16 in the momentum slots; FP32: word 7 = group coefficient, words 8-15 = 4 x {byte offset of Re J_k, coefficient};
// FP64: words 8-9 = group coefficient, words 12-27 = 4 x {offset, 0, coefficient}
template <typename T> struct TabCtl { unsigned ctl; T sg; bool chi; };

template <typename T> __device__ __forceinline__ cx<T> tab_dot(const cx<T>* a, const cx<T>* b) {      // Minkowski product, 2 MUL + 14 FMA
    cx<T> r;
    r.re = a[0].re * b[0].re - a[0].im * b[0].im - a[1].re * b[1].re + a[1].im * b[1].im - a[2].re * b[2].re + a[2].im * b[2].im - a[3].re * b[3].re + a[3].im * b[3].im;
    r.im = a[0].re * b[0].im + a[0].im * b[0].re - a[1].re * b[1].im - a[1].im * b[1].re - a[2].re * b[2].im - a[2].im * b[2].re - a[3].re * b[3].im - a[3].im * b[3].re;
    return r;
}
template <typename T> __device__ __forceinline__ cx<T> tab_kdot(const T* k1, const T* k2, const cx<T>* a) {       // (k1 - k2) . a
    const T d0 = k1[0] - k2[0], d1 = k1[1] - k2[1], d2 = k1[2] - k2[2], d3 = k1[3] - k2[3];
    return mk<T>(d0 * a[0].re - d1 * a[1].re - d2 * a[2].re - d3 * a[3].re, d0 * a[0].im - d1 * a[1].im - d2 * a[2].im - d3 * a[3].im);
}
template <typename T> __device__ __forceinline__ cx<T> tab_kvec(const T* d, const cx<T>* a) {
    return mk<T>(d[0] * a[0].re - d[1] * a[1].re - d[2] * a[2].re - d[3] * a[3].re, d[0] * a[0].im - d[1] * a[1].im - d[2] * a[2].im - d[3] * a[3].im);
}
// vvvxxx (eq. 24-27) with unit coupling: (a.b)((ka-kb).c) + (b.c)((kb-kc).a) + (c.a)((kc-ka).b)
template <typename T> __device__ __forceinline__ cx<T> tab_vvv(const TabOps<T>& O) {
    const cx<T>* a = O.w; const cx<T>* b = O.w + 4; const cx<T>* c = O.w + 8;
    const cx<T> ab = tab_dot<T>(a, b), bc = tab_dot<T>(b, c), ca = tab_dot<T>(c, a);
    // all momenta flow into the vertex, ka + kb + kc = 0:  kb - kc = ka + 2 kb,  kc - ka = -(2 ka + kb)
    T kbc[4], kca[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) { kbc[m] = O.k[m] + T(2) * O.k[4 + m]; kca[m] = -(T(2) * O.k[m] + O.k[4 + m]); }
    const cx<T> x = tab_kdot<T>(O.k, O.k + 4, c), y = tab_kvec<T>(kbc, a), z = tab_kvec<T>(kca, b);
    return mk<T>(ab.re * x.re - ab.im * x.im + bc.re * y.re - bc.im * y.im + ca.re * z.re - ca.im * z.im,
                 ab.re * x.im + ab.im * x.re + bc.re * y.im + bc.im * y.re + ca.re * z.im + ca.im * z.re);
}
// ggggxx (eqs. 32-36) with unit coupling, the piece being encoded in the operand order: (a.d)(b.c) - (a.c)(b.d)
template <typename T> __device__ __forceinline__ cx<T> tab_gggg(const TabOps<T>& O) {
    const cx<T>* a = O.w; const cx<T>* b = O.w + 4; const cx<T>* c = O.w + 8; const cx<T>* dd = O.w + 12;
    const cx<T> p = tab_dot<T>(a, dd), q = tab_dot<T>(b, c), r = tab_dot<T>(a, c), s = tab_dot<T>(b, dd);
    return mk<T>(p.re * q.re - p.im * q.im - r.re * s.re + r.im * s.im, p.re * q.im + p.im * q.re - r.re * s.im - r.im * s.re);
}
// iovxx0 (eqs. 18-22) with unit coupling
template <typename T> __device__ __forceinline__ cx<T> tab_iov(const TabOps<T>& O, T chi) {
    sp2<T> fi, fo; vec4<T> vc;
    fi.s[0] = O.w[0]; fi.s[1] = O.w[1]; fo.s[0] = O.w[2]; fo.s[1] = O.w[3];
    vc.v[0] = O.w[4]; vc.v[1] = O.w[5]; vc.v[2] = O.w[6]; vc.v[3] = O.w[7];
    return iovxx0<T>(fi, fo, vc, chi, T(1));
}

// ---- where a warp keeps its block of J (R complex numbers per lane) -----------------------------------------------------------
// JSmem: shared memory, element (k, re/im) of lane l at J[(2k + ri) * 32 + l].
// JTmem: tensor memory (TMEM, 256 kB per SM beside the 228 kB of shared memory): lane l of the warp's 32-lane quadrant, columns
//        2k, 2k+1 (FP32) or 4k..4k+3 (FP64), moved with tcgen05.ld / tcgen05.st (SASS: LDTM / STTM).  J is the largest per-warp
//        buffer (30 kB in FP32, 61 kB in FP64 for 120 colour elements): in TMEM it costs no shared memory, so twice as many warps
//        are resident for the processes whose J limited the occupancy, and its read-modify-write traffic leaves the LSU pipe.
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tm_ld2(unsigned ta, unsigned& a, unsigned& b) { asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];\n" : "=r"(a), "=r"(b) : "r"(ta)); }
__device__ __forceinline__ void tm_ld4(unsigned ta, unsigned& a, unsigned& b, unsigned& c, unsigned& d) { asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];\n" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(ta)); }
__device__ __forceinline__ void tm_st2(unsigned ta, unsigned a, unsigned b) { asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};\n" :: "r"(ta), "r"(a), "r"(b) : "memory"); }
__device__ __forceinline__ void tm_st4(unsigned ta, unsigned a, unsigned b, unsigned c, unsigned d) { asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};\n" :: "r"(ta), "r"(a), "r"(b), "r"(c), "r"(d) : "memory"); }

// turn passing between the warps of one block of J: mbarrier arrive = release, test / wait = acquire (no fence instruction on either side)
__device__ __forceinline__ void mb_init(unsigned a, unsigned count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"(a), "r"(count) : "memory"); }
__device__ __forceinline__ void mb_arrive(unsigned a) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" :: "r"(a) : "memory"); }
__device__ __forceinline__ bool mb_test(unsigned a, unsigned parity) {       // one look, no waiting
    unsigned ok;
    asm volatile("{\n.reg .pred P1;\nmbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\nselp.u32 %0, 1, 0, P1;\n}\n" : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void mb_wait(unsigned a, unsigned parity) {
    asm volatile("{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}\n" :: "r"(a), "r"(parity) : "memory");
}
template <typename T> __device__ __forceinline__ void q_put(unsigned char* p, T re, T im) {
    if constexpr (sizeof(T) == 4) *reinterpret_cast<float2*>(p) = make_float2(re, im); else cx_st<T>(p, mk<T>(re, im));
}
template <typename T> __device__ __forceinline__ void q_get(const unsigned char* p, T& re, T& im) {
    if constexpr (sizeof(T) == 4) { const float2 v = *reinterpret_cast<const float2*>(p); re = v.x; im = v.y; } else { const cx<T> v = cx_ld<T>(p); re = v.re; im = v.im; }
}
// shared-window address of the warp's FIFO block (0: the warp updates J at once); entries pushed so far
struct TabQueue { unsigned q; unsigned n; };

template <typename T> struct JSmem {
    T* J;
    __device__ __forceinline__ void zero(int R) { for (int a = 0; a < 2 * R; ++a) J[a * 32] = T(0); }
    // J_k += c_j (Sr, Si) for the nu <= 8 updates of a record; off = byte offset of Re J_k in the lane's column
    template <int NB> __device__ __forceinline__ void update(int nu, const unsigned* off, const T* c, T Sr, T Si) {
#pragma unroll
        for (int j = 0; j < HG_TAB_MAXU; ++j) if (j < nu) { T* pj = reinterpret_cast<T*>(reinterpret_cast<unsigned char*>(J) + off[j]); pj[0] += c[j] * Sr; pj[32] += c[j] * Si; }
    }
    // 8 consecutive elements starting at k0 (k0 a multiple of 8)
    __device__ __forceinline__ void block8(int k0, int R, T* xr, T* xi) {
#pragma unroll
        for (int i = 0; i < 8; ++i) { const bool in = k0 + i < R; xr[i] = in ? J[(2 * (k0 + i)) * 32] : T(0); xi[i] = in ? J[(2 * (k0 + i) + 1) * 32] : T(0); }
    }
};
template <typename T> struct JTmem {       // 8-byte elements: 4 columns per complex number
    unsigned ta;      // TMEM address of column 0 of this warp's block (lane field = first lane of the warp's quadrant)
    __device__ __forceinline__ void zero(int R) { for (int k = 0; k < (R + 7) / 8 * 8 + 1; ++k) tm_st4(ta + 4 * k, 0u, 0u, 0u, 0u); tm_wait_st(); }      // + the scratch element
    // NB updates in flight (4 NB registers): 2 keeps the closing loop inside its register budget, a FIFO drain affords 4.  The batches
    // are branch-free: the host pads every update list to a multiple of 4 with {scratch element, coefficient 0} (api.cu), so the
    // TMEM addresses of a batch move to uniform registers together instead of one R2UR at a time between branches
    template <int NB> __device__ __forceinline__ void update(int nu, const unsigned* off, const T* c, T Sr, T Si) {
        tm_wait_st();
#pragma unroll
        for (int j0 = 0; j0 < HG_TAB_MAXU; j0 += NB) {
            if (j0 >= nu) break;
            unsigned r[NB][4];
#pragma unroll
            for (int j = 0; j < NB; ++j) tm_ld4(ta + (off[j0 + j] >> 7), r[j][0], r[j][1], r[j][2], r[j][3]);
            tm_wait_ld();
#pragma unroll
            for (int j = 0; j < NB; ++j) {
                const T re = el<T>::from_bits(r[j][0], r[j][1]) + c[j0 + j] * Sr, im = el<T>::from_bits(r[j][2], r[j][3]) + c[j0 + j] * Si;
                tm_st4(ta + (off[j0 + j] >> 7), el<T>::lo(re), el<T>::hi(re), el<T>::lo(im), el<T>::hi(im));
            }
        }
    }
    __device__ __forceinline__ void block8(int k0, int, T* xr, T* xi) {
        tm_wait_st();
#pragma unroll
        for (int h = 0; h < 8; h += 4) {          // four complex numbers (16 registers) in flight
            unsigned r[4][4];
#pragma unroll
            for (int i = 0; i < 4; ++i) tm_ld4(ta + 4 * (k0 + h + i), r[i][0], r[i][1], r[i][2], r[i][3]);
            tm_wait_ld();
#pragma unroll
            for (int i = 0; i < 4; ++i) { xr[h + i] = el<T>::from_bits(r[i][0], r[i][1]); xi[h + i] = el<T>::from_bits(r[i][2], r[i][3]); }
        }
    }
};
template <> struct JTmem<float> {
    unsigned ta;
    __device__ __forceinline__ void zero(int R) { for (int k = 0; k < (R + 7) / 8 * 8 + 1; ++k) tm_st2(ta + 2 * k, 0u, 0u); tm_wait_st(); }
    template <int NB> __device__ __forceinline__ void update(int nu, const unsigned* off, const float* c, float Sr, float Si) {
        tm_wait_st();
#pragma unroll
        for (int j0 = 0; j0 < HG_TAB_MAXU; j0 += 2 * NB) {
            if (j0 >= nu) break;
            unsigned r[2 * NB][2];
#pragma unroll
            for (int j = 0; j < 2 * NB; ++j) tm_ld2(ta + (off[j0 + j] >> 7), r[j][0], r[j][1]);
            tm_wait_ld();
#pragma unroll
            for (int j = 0; j < 2 * NB; ++j) tm_st2(ta + (off[j0 + j] >> 7), __float_as_uint(__uint_as_float(r[j][0]) + c[j0 + j] * Sr), __float_as_uint(__uint_as_float(r[j][1]) + c[j0 + j] * Si));
        }
    }
    __device__ __forceinline__ void block8(int k0, int, float* xr, float* xi) {
        unsigned r[8][2];
        tm_wait_st();
#pragma unroll
        for (int i = 0; i < 8; ++i) tm_ld2(ta + 2 * (k0 + i), r[i][0], r[i][1]);
        tm_wait_ld();
#pragma unroll
        for (int i = 0; i < 8; ++i) { xr[i] = __uint_as_float(r[i][0]); xi[i] = __uint_as_float(r[i][1]); }
    }
};

// the update list of a record ({byte offset of Re J_k, coefficient} x 8), from the record itself or from a queue entry
template <typename T> __device__ __forceinline__ void tab_updates(const unsigned char* u, unsigned* off, T* c) {
    if constexpr (sizeof(T) == 4) {
#pragma unroll
        for (int j = 0; j < HG_TAB_MAXU; j += 2) { const uint4 v = *reinterpret_cast<const uint4*>(u + 8 * j); off[j] = v.x; c[j] = __uint_as_float(v.y); off[j + 1] = v.z; c[j + 1] = __uint_as_float(v.w); }
    } else {
#pragma unroll
        for (int j = 0; j < HG_TAB_MAXU; ++j) { const uint4 v = *reinterpret_cast<const uint4*>(u + 16 * j); off[j] = v.x; c[j] = el<T>::from_bits(v.z, v.w); }
    }
}
template <typename T> __device__ __forceinline__ const unsigned char* tab_rec_updates(const unsigned char* ent) { return ent + (sizeof(T) == 4 ? 32 : 48); }

// the amplitude goes into its group sum; at the end of a group, J_k += x_gk S_g (eq. 8) on the lane's column -- by this warp,
// or (several warps per block of J) later, when the warp's turn comes: S_g and the update list wait in the warp's FIFO
template <typename T, typename JP> __device__ __forceinline__ void tab_apply(const cx<T>& amp, const TabCtl<T>& C, const unsigned char* ent, JP& jp, T& Sr, T& Si, TabQueue& Q) {
    if ((C.ctl & 3u) != 3u) { Sr += C.sg * amp.re; Si += C.sg * amp.im; }
    const int nu = (C.ctl >> 3) & 15u;
    if (nu) {
        if (Q.q) {          // park the group sum and the record's update list in the warp's FIFO (the record loop keeps a slot free)
            const int lane = threadIdx.x & 31;
            unsigned char* qe = reinterpret_cast<unsigned char*>(__cvta_shared_to_generic(Q.q + HG_TAB_QHDR + (Q.n & (HG_TAB_QD - 1)) * tab_queue_bytes<T>()));
            q_put<T>(qe + lane * 2 * sizeof(T), Sr, Si);
            constexpr int UB = HG_TAB_MAXU * (sizeof(T) == 4 ? 8 : 16) / 16;      // 16-byte pieces of the update list
            if (lane < UB) *reinterpret_cast<uint4*>(qe + 32 * 2 * sizeof(T) + 16 + 16 * lane) = *reinterpret_cast<const uint4*>(tab_rec_updates<T>(ent) + 16 * lane);
            if (lane == UB) *reinterpret_cast<unsigned*>(qe + 32 * 2 * sizeof(T)) = (unsigned)nu | ((C.ctl & 4u) << 6);
            __syncwarp();
            ++Q.n;
        } else {
            unsigned off[HG_TAB_MAXU]; T c[HG_TAB_MAXU];
            tab_updates<T>(tab_rec_updates<T>(ent), off, c);
            jp.template update<2>(nu, off, c, Sr, Si);
        }
    }
    if (C.ctl & 4u) { Sr = T(0); Si = T(0); }
}

// One closing record from start to end.  The kind is tested ONCE and each branch loads its own operands, evaluates its vertex and
// applies the result, so no value has to be moved into common registers where the branches meet (such moves were 12 % of the
// instructions when the operands went through one shared structure).
template <typename T, typename JP> __device__ __forceinline__ void tab_record(const unsigned char* ent, const unsigned char* store, const T* evK, const unsigned char* myrows, JP& jp, T& Sr, T& Si, TabQueue& Q) {
    const uint4 q0 = *reinterpret_cast<const uint4*>(ent), q1 = *reinterpret_cast<const uint4*>(ent + 16);
    const unsigned kind = q0.x & 3u;
    TabCtl<T> C; C.ctl = q0.x;
    T sgc;
    if constexpr (sizeof(T) == 4) sgc = __uint_as_float(q1.w); else sgc = cx_ld<T>(ent + 32).re;
    const unsigned fb = myrows[q0.x >> 16];
    C.sg = (fb & 1u) ? sgc : T(0); C.chi = (fb & 2u) != 0u;
    if (kind == 3u) { tab_apply<T>(mk<T>(T(0), T(0)), C, ent, jp, Sr, Si, Q); return; }
    const unsigned aa = (q0.y & 0xffffu) + myrows[q0.w & 0xffffu], ab = (q0.y >> 16) + myrows[q0.w >> 16], ac = (q0.z & 0xffffu) + myrows[q1.x & 0xffffu];
    const unsigned sa = q1.y & 0xffu, sb = (q1.y >> 8) & 0xffu, sc = (q1.y >> 16) & 0xffu;
    if (kind == 0u) {
        TabOps<T> O;
        tab_ld<T>(O.w, store, aa, sa, 4); tab_ld<T>(O.w + 4, store, ab, sb, 4); tab_ld<T>(O.w + 8, store, ac, sc, 4);
        tab_ldk4<T>(O.k, reinterpret_cast<const T*>(reinterpret_cast<const unsigned char*>(evK) + (q1.z & 0xffffu)));
        tab_ldk4<T>(O.k + 4, reinterpret_cast<const T*>(reinterpret_cast<const unsigned char*>(evK) + (q1.z >> 16)));
        tab_apply<T>(tab_vvv<T>(O), C, ent, jp, Sr, Si, Q);
    } else if (kind == 1u) {
        TabOps<T> O;
        const unsigned ad = (q0.z >> 16) + myrows[q1.x >> 16], sd = q1.y >> 24;
        tab_ld<T>(O.w, store, aa, sa, 4); tab_ld<T>(O.w + 4, store, ab, sb, 4); tab_ld<T>(O.w + 8, store, ac, sc, 4); tab_ld<T>(O.w + 12, store, ad, sd, 4);
        tab_apply<T>(tab_gggg<T>(O), C, ent, jp, Sr, Si, Q);
    } else {
        TabOps<T> O;
        tab_ld<T>(O.w, store, aa, sa, 2); tab_ld<T>(O.w + 2, store, ab, sb, 2); tab_ld<T>(O.w + 4, store, ac, sc, 4);
        tab_apply<T>(tab_iov<T>(O, C.chi ? T(1) : T(-1)), C, ent, jp, Sr, Si, Q);
    }
}

// JM = 0: J in shared memory; JM = 1: J in tensor memory (tm_cols = columns this CTA allocates, tm_wcols = columns per warp).
// MW: several warps per block of J (FIFOs and turn passing compiled in); the one-warp kernels carry none of it.
// Register budget: the 8-byte element types get 136 with J in TMEM and one warp per J (at ptxas' default of 128 that instantiation
// spilled 4 bytes), 128 with several warps per J (so that FOUR warps per block of J, 16 per SM, fit the register file; the kernel
// forms its indices, its event number and its helicity weight again where phase C and the epilogue need them instead of carrying
// them through the closing loop, which is what it took to get there without a spill), 152 with J in shared memory; float gets 128.
// Zero local memory in all twelve instantiations.  The launch shape (api.cu, tab_pick_shape) keeps threads x registers inside the
// register file.
template <typename T, int JM, bool MW>
__global__ void __maxnreg__(sizeof(T) == 4 ? 128 : JM == 0 ? 152 : MW ? 128 : 136) k_tab(const TabDev d, const int epc, const int tm_cols, const int tm_wcols, const double* __restrict__ mom, const unsigned long long mom_stride, const unsigned long long n_events,
        const double inv_sqrt_s, const double out_scale, typename el<T>::out_t* __restrict__ me2, const int hel_mode, const int hel_fixed,
        const unsigned long long seed, const unsigned long long first_event) {
    typedef tabio<T> IO;
    extern __shared__ __align__(16) unsigned char hg_tab_smem[];
    // warps of a CTA: wic = sp * (epc * wpe) + slot * wpe + chunk.  The nsp warps with the same (slot, chunk) share that block of J:
    // wa = sp * wpe + chunk is the warp's index within its slot (nwe of them), te the thread's.
    // MW: several warps per block of J (d.nsp of them); the one-warp kernel carries none of the FIFO and turn-passing code
    const int n = d.n_ext, wpe = d.nchunks, nsp = MW ? d.nsp : 1, nwe = wpe * nsp, tpe = nwe * 32;
    const int tid = threadIdx.x, lane = tid & 31, wic = tid >> 5, W = epc * wpe, sp = wic / W, bw = wic - sp * W, el = bw / wpe, wie = bw - el * wpe, wa = sp * wpe + wie, te = wa * 32 + lane;
    // carve: [pm: double 4n x epc][red: double epc x wpe x 3 chains][per event: evK | evI | store][per (slot, chunk): J][per warp: ring][queues][rows]
    double* pm = reinterpret_cast<double*>(hg_tab_smem);
    double* red = pm + (size_t)4 * n * epc * hg::el<T>::EV;
    const size_t evb = tab_event_bytes<T>(d.nK, d.store32);
    unsigned char* evbase = reinterpret_cast<unsigned char*>(red + (size_t)epc * wpe * 3 * hg::el<T>::EV);
    evbase += (16 - ((size_t)(evbase - hg_tab_smem) & 15)) & 15;
    unsigned char* myev = evbase + (size_t)el * evb;
    T* evK = reinterpret_cast<T*>(myev);
    T* evI = evK + (size_t)4 * d.nK;
    unsigned char* store = myev + (size_t)d.nK * 4 * sizeof(T) + (((size_t)d.nK * sizeof(T) + 15) / 16) * 16;
    unsigned char* jbase = evbase + (size_t)epc * evb;
    const size_t jwb = JM ? 0 : tab_warp_bytes<T>(d.R);
    typename std::conditional<JM == 0, JSmem<T>, JTmem<T> >::type jp;
    if constexpr (JM == 0) jp.J = reinterpret_cast<T*>(jbase + (size_t)bw * jwb) + lane;
    unsigned char* ring = jbase + (size_t)epc * wpe * jwb + (size_t)wic * (HG_TAB_RING * tab_entry_bytes<T>());
    unsigned char* qbase = jbase + (size_t)epc * wpe * jwb + (size_t)epc * nwe * (HG_TAB_RING * tab_entry_bytes<T>());      // FIFOs: [block of J][warp]
    const int nq = nsp > 1 ? nsp : 0;                 // FIFOs (and turn barriers) per block of J
    unsigned char* rows = qbase + (size_t)W * nq * tab_qblock_bytes<T>();
    __shared__ unsigned int tm_base;
    for (int c = tid; c < W * nq; c += blockDim.x) mb_init((unsigned)__cvta_generic_to_shared(qbase + (size_t)c * tab_qblock_bytes<T>()), 32u);
    for (int c = tid; c < W * 3 * hg::el<T>::EV; c += blockDim.x) red[c] = 0.0;
    if constexpr (JM == 1) {
        // one warp allocates the CTA's TMEM columns and gives up the permit at once, so co-resident CTAs can allocate theirs
        if (tid < 32) {
            const unsigned dst = (unsigned)__cvta_generic_to_shared(&tm_base);
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" :: "r"(dst), "r"((unsigned)tm_cols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    }
    for (int c = tid; c < (d.n_rows * wpe * 32 + 3) / 4; c += blockDim.x) reinterpret_cast<unsigned int*>(rows)[c] = __ldg(reinterpret_cast<const unsigned int*>(d.lanerows) + c);

    // a slot of the CTA holds EV events (2 for the packed type: they travel in the two halves of every value)
    constexpr int EV = hg::el<T>::EV;
    const unsigned long long e0 = (unsigned long long)blockIdx.x * epc * EV;
    const unsigned long long e = e0 + (unsigned long long)el * EV;

#ifdef HG_TAB_TIMING
    long long tt0 = clock64(), tt1, tt2, tt3 = 0, tt4;
#endif
    const T* cf = reinterpret_cast<const T*>(d.coef);
    // ---- prologue ------------------------------------------------------------------------------------------------------
    const int epe = epc * EV;
    for (int c = tid; c < 4 * n * epe; c += blockDim.x) {
        unsigned long long ee = e0 + (unsigned long long)(c % epe); if (ee >= n_events) ee = n_events - 1;
        pm[c] = mom[(size_t)(c / epe) * mom_stride + ee] * inv_sqrt_s;
    }
    __syncthreads();
    if constexpr (JM == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
        // warp w of the CTA can reach TMEM lanes 32 (w % 4) .. +31 only; block bw of J sits in quadrant bw % 4, columns (bw / 4) tm_wcols .. ;
        // the warps that share it have the same w % 4 because epc * wpe is a multiple of 4 whenever nsp > 1 (api.cu, tab_pick_shape)
        jp.ta = tm_base + ((unsigned)((wic & 3) * 32) << 16) + (unsigned)((bw >> 2) * tm_wcols);
    }
    {
        typedef hg::el<T> EL;
        const double* pe = pm + el * EV;             // component c of the slot's event j: pe[c * epe + j]
        for (int s = te; s < d.nK; s += tpe) {       // momentum of a leg subset, all momenta flowing INTO the diagram, and 1/q^2
            const unsigned mask = __ldg(d.kmask + s);
            double k[2][4], iq[2];
#pragma unroll
            for (int j = 0; j < EV; ++j) {
                double k0 = 0, k1 = 0, k2 = 0, k3 = 0;
                for (int i = 0; i < n; ++i) if ((mask >> i) & 1u) {
                    const double sg = i < 2 ? 1.0 : -1.0;
                    k0 += sg * pe[(4 * i) * epe + j]; k1 += sg * pe[(4 * i + 1) * epe + j]; k2 += sg * pe[(4 * i + 2) * epe + j]; k3 += sg * pe[(4 * i + 3) * epe + j];
                }
                k[j][0] = k0; k[j][1] = k1; k[j][2] = k2; k[j][3] = k3;
                iq[j] = (mask & (mask - 1u)) ? 1.0 / (k0 * k0 - k1 * k1 - k2 * k2 - k3 * k3) : 0.0;
            }
            constexpr int J1 = EV - 1;
#pragma unroll
            for (int m = 0; m < 4; ++m) evK[4 * s + m] = EL::pack(k[0][m], k[J1][m]);
            evI[s] = EL::pack(iq[0], iq[J1]);
        }
        for (int i = te; i < n; i += tpe) {           // external wavefunctions, both helicities (variant 0: h = -1, variant 1: h = +1)
            const unsigned info = __ldg(d.leginfo + i), ty = info & 0xffu, base = info >> 16;
            constexpr int J1 = EV - 1;
            double b[2][6];
#pragma unroll
            for (int j = 0; j < EV; ++j) {
                const double p[4] = {pe[(4 * i) * epe + j], pe[(4 * i + 1) * epe + j], pe[(4 * i + 2) * epe + j], pe[(4 * i + 3) * epe + j]};
                if (ty < 2u) vxxxxx_basis<double>(p, ty == 1u, b[j], b[j] + 3); else ixxxxx_basis<double>(p, b[j]);
            }
            const unsigned single = (info >> 9) & 3u;      // 0: both helicities are stored (variants 0, 1); 1 / 2: the leg's helicity is -1 / +1 in every evaluated configuration
            if (ty < 2u) {
                const T rt[3] = {EL::pack(b[0][0], b[J1][0]), EL::pack(b[0][1], b[J1][1]), EL::pack(b[0][2], b[J1][2])};
                const T qt[3] = {EL::pack(b[0][3], b[J1][3]), EL::pack(b[0][4], b[J1][4]), EL::pack(b[0][5], b[J1][5])};
                if (single == 0u) { IO::stv(store, base, 1, vxxxxx<T>(rt, qt, T(-1))); IO::stv(store, base + 1, 1, vxxxxx<T>(rt, qt, T(1))); }
                else IO::stv(store, base, 0, vxxxxx<T>(rt, qt, single == 2u ? T(1) : T(-1)));
            } else {
                const T cs = ((info >> 8) & 1u) ? T(1) : T(-1);      // chirality = cs * helicity
                if constexpr (EV == 1) {
                    const T st3[3] = {EL::pack(b[0][0], 0.0), EL::pack(b[0][1], 0.0), EL::pack(b[0][2], 0.0)};
                    if (single == 0u) {
                        if (ty == 2u) { IO::sts(store, base, 1, ixxxxx<T>(st3, -cs)); IO::sts(store, base + 1, 1, ixxxxx<T>(st3, cs)); }
                        else          { IO::sts(store, base, 1, oxxxxx<T>(st3, -cs)); IO::sts(store, base + 1, 1, oxxxxx<T>(st3, cs)); }
                    } else {
                        const T ch = single == 2u ? cs : -cs;
                        if (ty == 2u) IO::sts(store, base, 0, ixxxxx<T>(st3, ch)); else IO::sts(store, base, 0, oxxxxx<T>(st3, ch));
                    }
                } else {
                    // the spinors of the two events are formed one by one (scalar FP32) and zipped: their construction branches on the chirality only
                    sp2<float> f[2][2];
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        const float st3[3] = {(float)b[j][0], (float)b[j][1], (float)b[j][2]};
                        const float c1 = ((info >> 8) & 1u) ? 1.f : -1.f;
                        if (ty == 2u) { f[j][0] = ixxxxx<float>(st3, -c1); f[j][1] = ixxxxx<float>(st3, c1); }
                        else          { f[j][0] = oxxxxx<float>(st3, -c1); f[j][1] = oxxxxx<float>(st3, c1); }
                    }
#pragma unroll
                    for (int v = 0; v < 2; ++v) {
                        if (single != 0u && v != (int)single - 1) continue;
                        sp2<T> z;
                        z.s[0] = mk<T>(EL::pack(f[0][v].s[0].re, f[1][v].s[0].re), EL::pack(f[0][v].s[0].im, f[1][v].s[0].im));
                        z.s[1] = mk<T>(EL::pack(f[0][v].s[1].re, f[1][v].s[1].re), EL::pack(f[0][v].s[1].im, f[1][v].s[1].im));
                        if (single == 0u) IO::sts(store, base + v, 1, z); else IO::sts(store, base, 0, z);
                    }
                }
            }
        }
    }
    if (sp == 0) {
        jp.zero(d.R);
        if constexpr (JM == 1) asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    }
    __syncthreads();
    if constexpr (JM == 1) asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");

#ifdef HG_TAB_TIMING
    tt1 = clock64();
#endif
    // ---- phase A: off-shell currents, once per helicity variant ----------------------------------------------------------
    for (int lev = 0; lev < d.n_levels; ++lev) {
        const int b1 = (int)__ldg(d.a_level + lev + 1);
        for (int b = (int)__ldg(d.a_level + lev) + wa; b < b1; b += nwe) {
            const uint4 hdr = __ldg(reinterpret_cast<const uint4*>(d.a_hdr) + b);
            const uint2 od = __ldg(reinterpret_cast<const uint2*>(d.a_out) + (size_t)b * 32 + lane);
            const int nt = hdr.x & 0xff, ptype = (hdr.x >> 8) & 0xff, t0 = hdr.x >> 16;
            const unsigned oaddr = od.x & 0xffffu, olnv = (od.x >> 16) & 7u; const bool active = (od.x >> 19) & 1u;
            const T inv = evI[od.y];
            if (ptype == 0) {
                vec4<T> acc;
#pragma unroll
                for (int m = 0; m < 4; ++m) acc.v[m] = mk<T>(T(0), T(0));
                for (int t = 0; t < nt; ++t) {
                    const uint4 td = __ldg(reinterpret_cast<const uint4*>(d.a_term) + (size_t)(t0 + t) * 32 + lane);
                    const unsigned kind = (hdr.y >> (4 * t)) & 15u;
                    const unsigned aa = td.x & 0xffffu, ab = td.x >> 16, ac = td.y & 0xffffu, la = (td.y >> 16) & 7u, lb = (td.y >> 19) & 7u, lc = (td.y >> 22) & 7u;
                    const T coef = cf[td.w];
                    if (kind == 0u) {
                        vacc(acc, jvvxx0<T>(IO::ldv(store, aa, la), IO::ldk(evK, td.z & 0xffu), IO::ldv(store, ab, lb), IO::ldk(evK, (td.z >> 8) & 0xffu), coef, inv));
                    } else if (kind == 1u) {
                        vacc(acc, jgggx0<T>(IO::ldv(store, aa, la), IO::ldv(store, ab, lb), IO::ldv(store, ac, lc), coef, inv));
                    } else {
                        const T chi = ((td.y >> 25) & 1u) ? T(1) : T(-1);
                        vacc(acc, jioxx0<T>(IO::lds(store, aa, la), IO::lds(store, ab, lb), chi, coef, inv));
                    }
                }
                if (active) IO::stv(store, oaddr, olnv, acc);
            } else {
                sp2<T> acc; acc.s[0] = mk<T>(T(0), T(0)); acc.s[1] = mk<T>(T(0), T(0));
                const mom4<T> ko = IO::ldk(evK, od.y);
                for (int t = 0; t < nt; ++t) {
                    const uint4 td = __ldg(reinterpret_cast<const uint4*>(d.a_term) + (size_t)(t0 + t) * 32 + lane);
                    const unsigned aa = td.x & 0xffffu, ab = td.x >> 16, la = (td.y >> 16) & 7u, lb = (td.y >> 19) & 7u;
                    const T coef = cf[td.w];
                    const T chi = ((td.y >> 25) & 1u) ? T(1) : T(-1);
                    if (ptype == 1) sacc(acc, fvixx0<T>(IO::lds(store, aa, la), IO::ldv(store, ab, lb), ko, chi, coef, inv));
                    else            sacc(acc, fvoxx0<T>(IO::lds(store, aa, la), IO::ldv(store, ab, lb), ko, chi, coef, inv));
                }
                if (active) IO::sts(store, oaddr, olnv, acc);
            }
        }
        __syncthreads();
    }

#ifdef HG_TAB_TIMING
    tt2 = clock64();
#endif
    // ---- phase B: closings, one helicity configuration per lane -------------------------------------------------------------
    // weight of the lane's configuration in the helicity sum, and whether this chunk of configurations has anything to do.  A lambda, called
    // before phase B (for chunk_on) and again in phase C (for the weight): nothing of it has to stay in a register through the closing loop.
    auto hel_weight = [&](int lane_, int wie_, unsigned long long e_, bool& on) {
        const int h = wie_ * d.cpc + lane_;
        const bool hvalid = lane_ < d.cpc && h < d.NH;
        T w = hvalid ? T(1) : T(0);
        on = true;
        if (hel_mode == 2) { w = (hvalid && h == hel_fixed) ? T(1) : T(0); on = hel_fixed >= wie_ * d.cpc && hel_fixed < (wie_ + 1) * d.cpc; }
        else if (hel_mode == 1) {
            double wj[2] = {0.0, 0.0}; on = false;
#pragma unroll
            for (int j = 0; j < EV; ++j) {
                unsigned int r[4]; unsigned long long ej = e_ + j; if (ej >= n_events) ej = n_events - 1;
                const unsigned long long ge = first_event + ej;
                philox4x32_10((unsigned int)ge, (unsigned int)(ge >> 32), 0xffffffffu, 0u, (unsigned int)seed, (unsigned int)(seed >> 32), r);
                const int hx = d.evalidx[r[0] >> (32 - n)];
                wj[j] = (hvalid && h == hx) ? (double)(1 << n) : 0.0;
                on = on || (hx >= wie_ * d.cpc && hx < (wie_ + 1) * d.cpc);
            }
            w = hg::el<T>::pack(wj[0], wj[EV - 1]);
        }
        return w;
    };
    bool chunk_on;
    (void)hel_weight(lane, wie, e, chunk_on);
    // The colour form is summed in THREE chains, chain c over the row tiles t = c mod 3, whatever the number of warps that share the
    // block of J: warp sp owns the chains with c mod min(nsp, 3) == sp.  A tile's contribution is reduced over the 32 lanes (helicity
    // sum, eq. 12, in the kernel's own precision: reading A21) and added to the chain in shared memory; the order of every addition is
    // the same for every launch shape, and so is the last bit of |M|^2.
    const int nown = nsp < 3 ? nsp : 3;
    if (chunk_on) {
        const int R = d.R;
        T Sr = T(0), Si = T(0);
        constexpr int ENT = tab_entry_bytes<T>(), NS = HG_TAB_RING;
        const unsigned char* myrows = rows + wie * 32 + lane;
        {
        const int nent = d.nrec[sp];                                  // this warp's list (padded with NS null records)
        const unsigned char* gent = d.b_ent + (size_t)d.list0[sp] * ENT;
        // Several warps per block of J: finished group sums wait in this warp's FIFO until the warp's turn comes.  Turn k of warp sp (its
        // groups k gpt .. k gpt + gpt - 1) follows turn k of warp sp - 1, or turn k - 1 of the last warp for sp = 0; a warp that completes a
        // turn arrives on its turn barrier with all lanes (after its TMEM stores have landed), the next warp looks at that barrier.
        TabQueue Q; Q.q = 0u; Q.n = 0u;
        unsigned applied = 0u, turn = 0u, prev = 0u;
        int gleft = 0;
        bool myturn = false;
        if constexpr (MW) {
            Q.q = (unsigned)__cvta_generic_to_shared(qbase + (size_t)(bw * nq + sp) * tab_qblock_bytes<T>());
            prev = (unsigned)__cvta_generic_to_shared(qbase + (size_t)(bw * nq + (sp == 0 ? nsp - 1 : sp - 1)) * tab_qblock_bytes<T>());
            gleft = d.ngrp[sp] < d.gpt ? d.ngrp[sp] : d.gpt;
            myturn = sp == 0;
        }
        // parity of the phase of the previous warp's barrier that turn `turn` of this warp waits for
        auto turn_parity = [&]() { return (sp == 0 ? turn - 1u : turn) & 1u; };
        // apply the parked groups for as long as it is this warp's turn
        auto drain = [&]() {
            if constexpr (JM == 1) asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
            while (applied != Q.n) {
                const unsigned char* qe = reinterpret_cast<const unsigned char*>(__cvta_shared_to_generic(Q.q + HG_TAB_QHDR + (applied & (HG_TAB_QD - 1)) * tab_queue_bytes<T>()));
                const unsigned hdr = *reinterpret_cast<const unsigned*>(qe + 32 * 2 * sizeof(T));
                unsigned off[HG_TAB_MAXU]; T c[HG_TAB_MAXU]; T gr, gi;
                q_get<T>(qe + lane * 2 * sizeof(T), gr, gi);
                tab_updates<T>(qe + 32 * 2 * sizeof(T) + 16, off, c);
                jp.template update<sizeof(T) == 4 ? 2 : 4>((int)(hdr & 0xffu), off, c, gr, gi);
                ++applied;
                if ((hdr & 0x100u) && --gleft == 0) {          // the turn is complete: pass it on
                    if constexpr (JM == 1) { tm_wait_st(); asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
                    mb_arrive(Q.q);
                    ++turn;
                    const int rest = d.ngrp[sp] - (int)turn * d.gpt;
                    gleft = rest < d.gpt ? rest : d.gpt;
                    myturn = gleft > 0 && mb_test(prev, turn_parity());
                    if (!myturn) break;
                    if constexpr (JM == 1) asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
                }
            }
        };
        // the closing records stream through a per-warp ring of 16 records in shared memory (cp.async), so the latency of the table
        // (L2) never shows.  refill: four records per cp.async group whenever no more than eight are ahead; after wait_group 1 every
        // record below issued - 4 has landed, and the loop never reads beyond that
        int issued = 0;
        auto refill = [&]() {
            const unsigned char* src = gent + (size_t)issued * ENT;
            unsigned char* dst = ring + (issued & (NS - 1)) * ENT;
#pragma unroll
            for (int q = 0; q < (4 * ENT + 511) / 512; ++q) {
                const int o = (q * 32 + lane) * 16;
                if (o < 4 * ENT) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"((unsigned)__cvta_generic_to_shared(dst + o)), "l"(src + o));
            }
            asm volatile("cp.async.commit_group;\n" ::);
            issued += 4;
        };
        static_assert(HG_TAB_RING == 16, "the refill logic assumes a ring of 16 records");
        refill(); refill(); refill();
        asm volatile("cp.async.wait_group 1;\n" ::); __syncwarp();
        // One closing at a time, one operand set in registers.  Measured and not adopted: fetching the next closing's operands while the current one is
        // computed (a second register set: C4 FP64 4.6e6 -> 3.1e6 events/s, the registers are worth more as resident warps), and
        // evaluating two neighbouring closings of one kind together for more instruction-level parallelism (C5 FP64 9.2e5 -> 8.4e5).
        for (int k = 0; k < nent; ++k) {
            if (issued - k <= 8) { refill(); asm volatile("cp.async.wait_group 1;\n" ::); __syncwarp(); }
            tab_record<T>(ring + (k & (NS - 1)) * ENT, store, evK, myrows, jp, Sr, Si, Q);
            if constexpr (MW) if (Q.n != applied) {                          // parked groups: is it this warp's turn?  (the FIFO must keep a slot free for the next record)
                if (!myturn) {
                    if (Q.n - applied == (unsigned)HG_TAB_QD) { mb_wait(prev, turn_parity()); myturn = true; }
                    else myturn = mb_test(prev, turn_parity());
                }
                if (myturn) drain();
            }
        }
        if constexpr (MW) while (Q.n != applied) {         // the rest of the parked groups
            if (!myturn) { mb_wait(prev, turn_parity()); myturn = true; }
            drain();
        }
        asm volatile("cp.async.wait_all;\n" ::);
        }
        if (nsp > 1) {          // J is complete when every warp that adds into it has had its last turn
            if constexpr (JM == 1) { tm_wait_st(); asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
            asm volatile("bar.sync %0, %1;\n" :: "r"(1 + bw), "r"(32 * nsp) : "memory");
            if constexpr (JM == 1) asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
        }
#ifdef HG_TAB_TIMING
        tt3 = clock64();
#endif
        // ---- phase C: colour form on the accumulated basis ----------------------------------------------------------------
        // (the thread's indices, its event and its weight are formed again here from a value the compiler cannot see through: kept in
        // registers through the closing loop they cost the 128-register kernels a spill)
        int tid_c = threadIdx.x; asm volatile("" : "+r"(tid_c));
        const int lane = tid_c & 31, wic = tid_c >> 5, sp = wic / W, bw = wic - sp * W, el = bw / wpe, wie = bw - el * wpe;
        const unsigned long long e = ((unsigned long long)blockIdx.x * epc + (unsigned long long)el) * EV;
        double* red = reinterpret_cast<double*>(hg_tab_smem) + (size_t)4 * n * epc * EV;
        bool on_c; const T wgt = hel_weight(lane, wie, e, on_c); (void)on_c;
        // t_a = C_aa J_a + sum_{b > a} 2 C_ab J_b for a tile of 8 rows stays in registers while J streams through (from shared
        // memory or TMEM) in blocks of 8 columns.  The 8 x 8 coefficient block of each step comes through the warp's ring
        // (free after phase B) by cp.async, one block ahead, so the latency of the matrix (L2) is hidden.
        const T* cm = reinterpret_cast<const T*>(d.cmat);
        const int ntile = d.Rpad / 8;
        if (d.cstage == 3) {
            // hand J to the tensor-core colour kernel: one row per (event, configuration, re/im), Rpad columns, written 8 at a time
            typedef typename hg::el<T>::out_t OT;
            OT* X = reinterpret_cast<OT*>(d.jout);
            for (int bb = sp; bb < ntile; bb += nsp) {
                T xr[8], xi[8];
                jp.block8(8 * bb, R, xr, xi);
#pragma unroll
                for (int j = 0; j < EV; ++j) {
                    if (e + j >= n_events) continue;
                    OT* row = X + ((((size_t)(e + j) * wpe + wie) * 32 + lane) * 2) * d.Rpad + 8 * bb;
#pragma unroll
                    for (int i = 0; i < 8; ++i) { row[i] = hg::el<T>::half(xr[i], j); row[d.Rpad + i] = hg::el<T>::half(xi[i], j); }
                }
            }
        } else {
        constexpr int CB = 64 * sizeof(T);                    // bytes of one coefficient block
        __syncwarp();
        const int cstage = d.cstage;
        const T* cvals = reinterpret_cast<const T*>(d.cvals);
        auto fetch = [&](int t, int bb, int buf) {
            const size_t blk = ((size_t)t * d.Rpad + (size_t)8 * bb) * 8;        // first coefficient of the block
            if (t < ntile) {
                if (cstage == 1) {                // 64 one-byte indices
                    if (lane < 4) {
                        const unsigned dst = (unsigned)__cvta_generic_to_shared(ring + buf * CB + lane * 16);
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(dst), "l"(d.cidx + blk + lane * 16));
                    }
                } else if (lane < CB / 16) {
                    const unsigned dst = (unsigned)__cvta_generic_to_shared(ring + buf * CB + lane * 16);
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(dst), "l"(reinterpret_cast<const unsigned char*>(cm + blk) + lane * 16));
                }
            }
            asm volatile("cp.async.commit_group;\n" ::);
        };
        int buf = 0;
        // row tiles of this warp: those of the chains it owns, in increasing order
        auto next_tile = [&](int t) { ++t; while (t < ntile && (t % 3) % nown != sp) ++t; return t; };
        int t = next_tile(-1);
        fetch(t, t, 0);
        for (; t < ntile; t = next_tile(t)) {
            T tr[8], ti[8], dr[8], di[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) { tr[i] = T(0); ti[i] = T(0); }
            for (int bb = t; bb < ntile; ++bb) {
                // next block: (t, bb + 1), or the first block of the next tile (nothing after the last one: an empty group)
                const bool last_bb = bb + 1 == ntile;
                const int tn = last_bb ? next_tile(t) : t;
                fetch(tn, last_bb ? tn : bb + 1, buf ^ 1);
                T xr[8], xi[8];
                jp.block8(8 * bb, R, xr, xi);
                if (bb == t) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) { dr[i] = xr[i]; di[i] = xi[i]; }
                }
                asm volatile("cp.async.wait_group 1;\n" ::); __syncwarp();
                const T* cblk = reinterpret_cast<const T*>(ring + buf * CB);
                if (cstage == 1) {
                    // the paper's colour stage: only the distinct values of the matrix are stored, an index map says
                    // which one sits where
                    const unsigned char* iblk = ring + buf * CB;
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const uint2 ib = *reinterpret_cast<const uint2*>(iblk + q * 8);
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            const T c = cvals[((i < 4 ? ib.x : ib.y) >> (8 * (i & 3))) & 0xffu];
                            tr[i] += c * xr[q]; ti[i] += c * xi[q];
                        }
                    }
                } else {
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    T c8[8];
                    if constexpr (sizeof(T) == 4) {
                        const float4 c0 = *reinterpret_cast<const float4*>(cblk + q * 8), c1 = *reinterpret_cast<const float4*>(cblk + q * 8 + 4);
                        c8[0] = c0.x; c8[1] = c0.y; c8[2] = c0.z; c8[3] = c0.w; c8[4] = c1.x; c8[5] = c1.y; c8[6] = c1.z; c8[7] = c1.w;
                    } else {
                        const uint4* rp = reinterpret_cast<const uint4*>(cblk + q * 8);
#pragma unroll
                        for (int i = 0; i < 4; ++i) { const cx<T> u = cx_ld<T>(rp + i); c8[2 * i] = u.re; c8[2 * i + 1] = u.im; }
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) { tr[i] += c8[i] * xr[q]; ti[i] += c8[i] * xi[q]; }
                }
                }
                __syncwarp();
                buf ^= 1;
            }
            T ft = T(0);
            if (cstage == 2) {        // tiles of the Cholesky factor: t_k = sum_{b >= k} L_bk J_b, form = sum_k |t_k|^2
#pragma unroll
                for (int i = 0; i < 8; ++i) ft += tr[i] * tr[i] + ti[i] * ti[i];
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) ft += dr[i] * tr[i] + di[i] * ti[i];
            }
            ft = wgt * ft;
#pragma unroll
            for (int j = 0; j < EV; ++j) {
                typename hg::el<T>::out_t a = hg::el<T>::half(ft, j);
                for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                if (lane == 0) { double* rc = red + ((size_t)(bw * 3 + t % 3) * EV + j); *rc = (double)((typename hg::el<T>::out_t)*rc + a); }
            }
        }
        asm volatile("cp.async.wait_all;\n" ::);
        }
    }
    // ---- helicity sum (eq. 12) and averaging factors -------------------------------------------------------------
#ifdef HG_TAB_TIMING      // debug build only: cycles per phase, summed over warps
    tt4 = clock64();
    if (lane == 0 && chunk_on) { atomicAdd(&g_tab_timing[0], (unsigned long long)(tt1 - tt0)); atomicAdd(&g_tab_timing[1], (unsigned long long)(tt2 - tt1)); atomicAdd(&g_tab_timing[2], (unsigned long long)(tt3 - tt2)); atomicAdd(&g_tab_timing[3], (unsigned long long)(tt4 - tt3)); atomicAdd(&g_tab_timing[4], 1ull); }
#endif
    if constexpr (JM == 1) { tm_wait_ld(); tm_wait_st(); asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
    __syncthreads();
    int tid_e = threadIdx.x; asm volatile("" : "+r"(tid_e));          // again: indices formed where they are used
    const int wic_e = tid_e >> 5, sp_e = wic_e / W, bw_e = wic_e - sp_e * W, el_e = bw_e / wpe, te_e = (sp_e * wpe + bw_e - el_e * wpe) * 32 + (tid_e & 31);
    const unsigned long long e_e = ((unsigned long long)blockIdx.x * epc + (unsigned long long)el_e) * EV;
    const double* red_e = reinterpret_cast<const double*>(hg_tab_smem) + (size_t)4 * n * epc * EV;
    if (te_e < EV && e_e + te_e < n_events && d.cstage != 3) {
        typedef typename hg::el<T>::out_t OT;
        OT s = 0;           // chains and chunks in a fixed order
        for (int w = 0; w < wpe; ++w) { const double* r3 = red_e + (size_t)((el_e * wpe + w) * 3) * EV + te_e; s += ((OT)r3[0] + (OT)r3[EV]) + (OT)r3[2 * EV]; }
        me2[e_e + te_e] = (typename hg::el<T>::out_t)(out_scale * (double)s);
    }
    if constexpr (JM == 1) {
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(tm_base), "r"((unsigned)tm_cols) : "memory");
    }
}
#endif

}  // namespace hg
