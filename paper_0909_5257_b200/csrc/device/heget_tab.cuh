// heget-b200: the TABLE-DRIVEN evaluator of steps a3-a8 (eq. 4) -- one generic kernel per
// precision that interprets the table program the generator (csrc/gen/tab.hpp) writes for a process.  No per-process code:
// the whole kernel is a few kB of instructions, so the instruction cache holds it (the straight-line kernels of the big
// processes were instruction-fetch bound).
//
// Work decomposition (one CTA = EPC events x WPE warps, WPE = ceil(n_hel_eval / 32)):
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
//   phase C   colour form  Jr^T C Jr + Ji^T C Ji (eq. 10) per lane, register-tiled over 8 rows, C streamed from
//             global memory (L1 broadcasts); helicity sum (eq. 12) by warp shuffles; me2 = out_scale * sum.
// Current store layout: 16-byte chunks; a current with nv variants and ncomp complex components occupies
// chunk(q, v) = base + q * nv + v, each chunk holding 2 complex (FP32) or 1 complex (FP64) -- lanes that share a variant read
// the same chunk (multicast), lanes with different variants read neighbouring chunks (no bank conflict).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "heget_dev.cuh"
#include "heget_rt.cuh"

namespace hg {

struct TabDev {
    int n_ext, NH, nchunks, cpc, R, Rpad, nK, store32, n_levels, n_closings;
    const uint32_t* kmask; const uint32_t* leginfo;
    const uint32_t* a_hdr; const uint32_t* a_out; const uint32_t* a_term; const uint32_t* a_level;
    const uint32_t* b_entry; const uint32_t* b_vtab;
    const uint16_t* jl_index; const uint16_t* jl_coef;
    const void* coef;            // T[]: pool of rational coefficients
    const void* cmat;            // T[(Rpad/8) * R * 8]
    const short* evalidx;        // [2^n_ext] helicity bits -> evaluated configuration or -1
};

// shared-memory bytes of one event (momenta slots + store) and of one warp's J column block
template <typename T> __host__ __device__ inline size_t tab_event_bytes(int nK, int store32) {
    return (size_t)nK * 4 * sizeof(T) + (((size_t)nK * sizeof(T) + 15) / 16) * 16 + (size_t)store32 * 16 * (sizeof(T) / 4);
}
template <typename T> __host__ __device__ inline size_t tab_warp_bytes(int R) { return (size_t)2 * R * 32 * sizeof(T); }
template <typename T> inline size_t tab_smem_bytes(const TabDev& d, int epc) {
    return (size_t)epc * (sizeof(double) * 4 * d.n_ext + tab_event_bytes<T>(d.nK, d.store32) + (size_t)d.nchunks * tab_warp_bytes<T>(d.R) + sizeof(double) * d.nchunks);
}

#if defined(__CUDACC__)
template <typename T> struct tabio;
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
template <> struct tabio<double> {
    // FP64 chunk of (current base32 b, variant v): 2 b + q nv + v; addr = b + v with b a multiple of nv
    static __device__ __forceinline__ unsigned a64(unsigned addr, unsigned lnv) { const unsigned m = (1u << lnv) - 1u; return 2u * (addr & ~m) + (addr & m); }
    static __device__ __forceinline__ vec4<double> ldv(const unsigned char* st, unsigned addr, unsigned lnv) {
        const double2* s = reinterpret_cast<const double2*>(st) + a64(addr, lnv);
        const unsigned nv = 1u << lnv;
        const double2 c0 = s[0], c1 = s[nv], c2 = s[2 * nv], c3 = s[3 * nv];
        vec4<double> w; w.v[0] = mk<double>(c0.x, c0.y); w.v[1] = mk<double>(c1.x, c1.y); w.v[2] = mk<double>(c2.x, c2.y); w.v[3] = mk<double>(c3.x, c3.y); return w;
    }
    static __device__ __forceinline__ void stv(unsigned char* st, unsigned addr, unsigned lnv, const vec4<double>& w) {
        double2* s = reinterpret_cast<double2*>(st) + a64(addr, lnv);
        const unsigned nv = 1u << lnv;
        s[0] = make_double2(w.v[0].re, w.v[0].im); s[nv] = make_double2(w.v[1].re, w.v[1].im); s[2 * nv] = make_double2(w.v[2].re, w.v[2].im); s[3 * nv] = make_double2(w.v[3].re, w.v[3].im);
    }
    static __device__ __forceinline__ sp2<double> lds(const unsigned char* st, unsigned addr, unsigned lnv) {
        const double2* s = reinterpret_cast<const double2*>(st) + a64(addr, lnv);
        const double2 c0 = s[0], c1 = s[1u << lnv];
        sp2<double> f; f.s[0] = mk<double>(c0.x, c0.y); f.s[1] = mk<double>(c1.x, c1.y); return f;
    }
    static __device__ __forceinline__ void sts(unsigned char* st, unsigned addr, unsigned lnv, const sp2<double>& f) {
        double2* s = reinterpret_cast<double2*>(st) + a64(addr, lnv);
        s[0] = make_double2(f.s[0].re, f.s[0].im); s[1u << lnv] = make_double2(f.s[1].re, f.s[1].im);
    }
    static __device__ __forceinline__ mom4<double> ldk(const double* evk, unsigned slot) {
        const double2* s = reinterpret_cast<const double2*>(evk) + 2 * slot;
        const double2 c0 = s[0], c1 = s[1];
        mom4<double> k; k.p[0] = c0.x; k.p[1] = c0.y; k.p[2] = c1.x; k.p[3] = c1.y; return k;
    }
};

template <typename T> __device__ __forceinline__ void vacc(vec4<T>& a, const vec4<T>& b) {
#pragma unroll
    for (int m = 0; m < 4; ++m) { a.v[m].re += b.v[m].re; a.v[m].im += b.v[m].im; }
}
template <typename T> __device__ __forceinline__ void sacc(sp2<T>& a, const sp2<T>& b) {
    a.s[0].re += b.s[0].re; a.s[0].im += b.s[0].im; a.s[1].re += b.s[1].re; a.s[1].im += b.s[1].im;
}

template <typename T>
__global__ void __launch_bounds__(256) k_tab(const TabDev d, const int epc, const double* __restrict__ mom, const unsigned long long n_events,
        const double inv_sqrt_s, const double out_scale, T* __restrict__ me2, const int hel_mode, const int hel_fixed,
        const unsigned long long seed, const unsigned long long first_event) {
    typedef tabio<T> IO;
    extern __shared__ __align__(16) unsigned char hg_tab_smem[];
    const int n = d.n_ext, wpe = d.nchunks, tpe = wpe * 32;
    const int tid = threadIdx.x, el = tid / tpe, te = tid % tpe, wie = te >> 5, lane = tid & 31;
    // carve: [pm: double 4n x epc][red: double epc x wpe][per event: evK | evI | store][per warp: J]
    double* pm = reinterpret_cast<double*>(hg_tab_smem);
    double* red = pm + (size_t)4 * n * epc;
    const size_t evb = tab_event_bytes<T>(d.nK, d.store32);
    unsigned char* evbase = reinterpret_cast<unsigned char*>(red + (size_t)epc * wpe);
    evbase += (16 - ((size_t)(evbase - hg_tab_smem) & 15)) & 15;
    unsigned char* myev = evbase + (size_t)el * evb;
    T* evK = reinterpret_cast<T*>(myev);
    T* evI = evK + (size_t)4 * d.nK;
    unsigned char* store = myev + (size_t)d.nK * 4 * sizeof(T) + (((size_t)d.nK * sizeof(T) + 15) / 16) * 16;
    T* J = reinterpret_cast<T*>(evbase + (size_t)epc * evb + (size_t)(el * wpe + wie) * tab_warp_bytes<T>(d.R)) + lane;

    const unsigned long long e0 = (unsigned long long)blockIdx.x * epc;
    unsigned long long e = e0 + el;
    const bool live = e < n_events;
    if (!live) e = n_events - 1;

    const T* cf = reinterpret_cast<const T*>(d.coef);
    // ---- prologue ------------------------------------------------------------------------------------------------------
    for (int c = tid; c < 4 * n * epc; c += blockDim.x) {
        unsigned long long ee = e0 + (unsigned long long)(c % epc); if (ee >= n_events) ee = n_events - 1;
        pm[c] = mom[(size_t)(c / epc) * n_events + ee] * inv_sqrt_s;
    }
    __syncthreads();
    {
        const double* pe = pm + el;
        for (int s = te; s < d.nK; s += tpe) {       // momentum of a leg subset, all momenta flowing INTO the diagram, and 1/q^2
            const unsigned mask = __ldg(d.kmask + s);
            double k0 = 0, k1 = 0, k2 = 0, k3 = 0;
            for (int i = 0; i < n; ++i) if ((mask >> i) & 1u) {
                const double sg = i < 2 ? 1.0 : -1.0;
                k0 += sg * pe[(4 * i) * epc]; k1 += sg * pe[(4 * i + 1) * epc]; k2 += sg * pe[(4 * i + 2) * epc]; k3 += sg * pe[(4 * i + 3) * epc];
            }
            evK[4 * s] = (T)k0; evK[4 * s + 1] = (T)k1; evK[4 * s + 2] = (T)k2; evK[4 * s + 3] = (T)k3;
            evI[s] = (mask & (mask - 1u)) ? (T)(1.0 / (k0 * k0 - k1 * k1 - k2 * k2 - k3 * k3)) : T(0);
        }
        for (int i = te; i < n; i += tpe) {           // external wavefunctions, both helicities (variant 0: h = -1, variant 1: h = +1)
            const unsigned info = __ldg(d.leginfo + i), ty = info & 0xffu, base = info >> 16;
            const double p[4] = {pe[(4 * i) * epc], pe[(4 * i + 1) * epc], pe[(4 * i + 2) * epc], pe[(4 * i + 3) * epc]};
            if (ty < 2u) {
                double r[3], q[3]; vxxxxx_basis<double>(p, ty == 1u, r, q);
                const T rt[3] = {(T)r[0], (T)r[1], (T)r[2]}, qt[3] = {(T)q[0], (T)q[1], (T)q[2]};
                IO::stv(store, base, 1, vxxxxx<T>(rt, qt, T(-1))); IO::stv(store, base + 1, 1, vxxxxx<T>(rt, qt, T(1)));
            } else {
                double s3[3]; ixxxxx_basis<double>(p, s3);
                const T st3[3] = {(T)s3[0], (T)s3[1], (T)s3[2]};
                const T cs = ((info >> 8) & 1u) ? T(1) : T(-1);      // chirality = cs * helicity
                if (ty == 2u) { IO::sts(store, base, 1, ixxxxx<T>(st3, -cs)); IO::sts(store, base + 1, 1, ixxxxx<T>(st3, cs)); }
                else          { IO::sts(store, base, 1, oxxxxx<T>(st3, -cs)); IO::sts(store, base + 1, 1, oxxxxx<T>(st3, cs)); }
            }
        }
    }
    __syncthreads();

    // ---- phase A: off-shell currents, once per helicity variant ----------------------------------------------------------
    for (int lev = 0; lev < d.n_levels; ++lev) {
        const int b1 = (int)__ldg(d.a_level + lev + 1);
        for (int b = (int)__ldg(d.a_level + lev) + wie; b < b1; b += wpe) {
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
                    const T coef = __ldg(cf + td.w);
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
                    const T coef = __ldg(cf + td.w);
                    const T chi = ((td.y >> 25) & 1u) ? T(1) : T(-1);
                    if (ptype == 1) sacc(acc, fvixx0<T>(IO::lds(store, aa, la), IO::ldv(store, ab, lb), ko, chi, coef, inv));
                    else            sacc(acc, fvoxx0<T>(IO::lds(store, aa, la), IO::ldv(store, ab, lb), ko, chi, coef, inv));
                }
                if (active) IO::sts(store, oaddr, olnv, acc);
            }
        }
        __syncthreads();
    }

    // ---- phase B: closings, one helicity configuration per lane -------------------------------------------------------------
    const int h = wie * d.cpc + lane;
    const bool hvalid = lane < d.cpc && h < d.NH;
    T wgt = hvalid ? T(1) : T(0);
    bool chunk_on = true;
    if (hel_mode == 2) { wgt = (hvalid && h == hel_fixed) ? T(1) : T(0); chunk_on = hel_fixed >= wie * d.cpc && hel_fixed < (wie + 1) * d.cpc; }
    else if (hel_mode == 1) {
        unsigned int r[4]; const unsigned long long ge = first_event + e;
        philox4x32_10((unsigned int)ge, (unsigned int)(ge >> 32), 0xffffffffu, 0u, (unsigned int)seed, (unsigned int)(seed >> 32), r);
        const int hx = d.evalidx[r[0] >> (32 - n)];
        wgt = (hvalid && h == hx) ? T(1 << n) : T(0); chunk_on = hx >= wie * d.cpc && hx < (wie + 1) * d.cpc;
    }
    T form = T(0);
    if (chunk_on) {
        const int R = d.R;
        for (int a = 0; a < 2 * R; ++a) J[a * 32] = T(0);
        T Sr = T(0), Si = T(0);
        const uint32_t* vt = d.b_vtab + (size_t)wie * 32 + lane;
        const int stride = wpe * 32;
        for (int k = 0; k < d.n_closings; ++k) {
            const uint4 e0w = __ldg(reinterpret_cast<const uint4*>(d.b_entry) + 2 * k);
            const uint2 e1w = __ldg(reinterpret_cast<const uint2*>(d.b_entry) + 4 * k + 2);
            const unsigned w = __ldg(vt + (size_t)k * stride);
            const unsigned ba = e0w.x & 0xffffu, bb = e0w.x >> 16, bc = e0w.y & 0xffffu, bd = e0w.y >> 16;
            const unsigned la = e0w.z & 7u, lb = (e0w.z >> 3) & 7u, lc = (e0w.z >> 6) & 7u, ld = (e0w.z >> 9) & 7u, kind = (e0w.z >> 12) & 7u;
            const unsigned va = w & 31u, vb = (w >> 5) & 31u, vc = (w >> 10) & 31u, vd = (w >> 15) & 31u;
            cx<T> amp;
            if (kind == 0u) {
                amp = vvvxxx<T>(IO::ldv(store, ba + va, la), IO::ldk(evK, (e0w.z >> 16) & 0xffu), IO::ldv(store, bb + vb, lb), IO::ldk(evK, e0w.z >> 24),
                                IO::ldv(store, bc + vc, lc), IO::ldk(evK, e0w.w & 0xffu), T(1));
            } else if (kind == 1u) {
                amp = ggggxx<T>(IO::ldv(store, ba + va, la), IO::ldv(store, bb + vb, lb), IO::ldv(store, bc + vc, lc), IO::ldv(store, bd + vd, ld), T(1));
            } else {
                const T chi = ((w >> 20) & 1u) ? T(1) : T(-1);
                amp = iovxx0<T>(IO::lds(store, ba + va, la), IO::lds(store, bb + vb, lb), IO::ldv(store, bc + vc, lc), chi, T(1));
            }
            const T sg = ((w >> 21) & 1u) ? __ldg(cf + e1w.x) : T(0);
            Sr += sg * amp.re; Si += sg * amp.im;
            if ((e0w.z >> 15) & 1u) {
                const int jc = (e0w.w >> 8) & 0xff; const unsigned jo = e1w.y;
                for (int j = 0; j < jc; ++j) {
                    const int idx = __ldg(d.jl_index + jo + j); const T c = __ldg(cf + __ldg(d.jl_coef + jo + j));
                    J[(2 * idx) * 32] += c * Sr; J[(2 * idx + 1) * 32] += c * Si;
                }
                Sr = T(0); Si = T(0);
            }
        }
        // ---- phase C: colour form on the accumulated basis ----------------------------------------------------------------
        const T* cm = reinterpret_cast<const T*>(d.cmat);
        for (int t = 0; t < d.Rpad / 8; ++t) {
            T tr[8], ti[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) { tr[i] = T(0); ti[i] = T(0); }
            const T* row = cm + (size_t)t * R * 8;
            for (int b = 8 * t; b < R; ++b) {
                const T xr = J[(2 * b) * 32], xi = J[(2 * b + 1) * 32];
                T c8[8];
                if constexpr (sizeof(T) == 4) {
                    const float4 c0 = __ldg(reinterpret_cast<const float4*>(row + (size_t)b * 8)), c1 = __ldg(reinterpret_cast<const float4*>(row + (size_t)b * 8) + 1);
                    c8[0] = c0.x; c8[1] = c0.y; c8[2] = c0.z; c8[3] = c0.w; c8[4] = c1.x; c8[5] = c1.y; c8[6] = c1.z; c8[7] = c1.w;
                } else {
                    const double2* rp = reinterpret_cast<const double2*>(row + (size_t)b * 8);
                    const double2 c0 = __ldg(rp), c1 = __ldg(rp + 1), c2 = __ldg(rp + 2), c3 = __ldg(rp + 3);
                    c8[0] = c0.x; c8[1] = c0.y; c8[2] = c1.x; c8[3] = c1.y; c8[4] = c2.x; c8[5] = c2.y; c8[6] = c3.x; c8[7] = c3.y;
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) { tr[i] += c8[i] * xr; ti[i] += c8[i] * xi; }
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) if (8 * t + i < R) form += J[(2 * (8 * t + i)) * 32] * tr[i] + J[(2 * (8 * t + i) + 1) * 32] * ti[i];
        }
    }
    // ---- helicity sum (eq. 12) and averaging factors -------------------------------------------------------------
    double acc = (double)(wgt * form);
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) red[el * wpe + wie] = acc;
    __syncthreads();
    if (te == 0 && live) {
        double s = 0; for (int w = 0; w < wpe; ++w) s += red[el * wpe + w];
        me2[e] = (T)(out_scale * s);
    }
}
#endif

}  // namespace hg
