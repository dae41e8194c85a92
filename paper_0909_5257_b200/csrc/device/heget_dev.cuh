// heget-b200 device library: HELAS-style wavefunctions and vertex functions for massless QCD,
// templated on the arithmetic type T (double = FP64 path, float = FP32 path).
//
// PAPER.md:217-389 (section 4) names the functions; the paper's listings are empty/garbled in the extraction
// (PAPER.md:489-533), so every body below is written from the Lagrangian terms the paper prints:
//   L_qqg  = -g T^a A^a_mu qbar gamma^mu q                     eq. 19
//   L_ggg  =  g f^{abc} (d^mu A^{a nu}) A^b_mu A^c_nu          eq. 23
//   L_gggg = -g^2/4 f^{abe} f^{cde} A^{a mu} A^{b nu} A^c_mu A^d_nu   eq. 31
// with the paper's colour-factor conventions: -T^a per quark-gluon vertex (eq. 22), i f^{abc} per
// three-gluon vertex (eqs. 27, 30), f^{abe}f^{cde}, f^{ace}f^{dbe}, f^{ade}f^{bce} for the three
// four-gluon pieces (eqs. 36, 40).  With those colour factors pulled out, and one overall i per
// diagram dropped (it is the same for every diagram), every function has REAL coefficients:
//   gluon line from ggg vertex + Feynman-gauge propagator:   + g V3 / q^2
//   gluon line from gggg vertex + propagator:                - g^2 W_piece / q^2
//   gluon line from a quark pair:                                           + g (psibar gamma^mu psi) / q^2
//   quark line after absorbing a gluon (massless propagator):               - g kslash epsslash psi / k^2
//   closing vertices (no propagator):   + g V3,  - g^2 W_piece,  + g psibar epsslash psi.
//
// Differences from the paper's HEGET (design for B200):
//  * a wavefunction does NOT carry its momentum in slots [4],[5]: momenta of leg subsets are
//    helicity independent, so they live once per event as real 4-vectors and are passed separately;
//  * 1/q^2 is passed in (computed once per event, not once per helicity);
//  * massless quark lines conserve chirality, so fermion wavefunctions are 2-component Weyl spinors plus the line's
//    chirality sign chi (+1: left-handed line, -1: right-handed line) instead of cmplx[6] with two zero entries.
// Metric (+,-,-,-); 4-vectors are (E, x, y, z) with UPPER indices; all momenta flow INTO the diagram.
#pragma once
#include <cstring>

#if defined(__CUDACC__)
#define HG_HD __host__ __device__ __forceinline__
#else
#define HG_HD inline
#endif

// vertex-level functions: inlined into the generated body by default; -DHG_CALL_VERTEX makes them real calls so that a long
// body holds one copy of each (an experiment against the instruction-fetch bound of the big processes)
#if defined(HG_CALL_VERTEX) && defined(__CUDACC__)
#define HG_VX __device__ __noinline__
#define HG_CV4 const vec4<T>
#define HG_CM4 const mom4<T>
#define HG_CS2 const sp2<T>
#else
#define HG_VX HG_HD
#define HG_CV4 const vec4<T>&
#define HG_CM4 const mom4<T>&
#define HG_CS2 const sp2<T>&
#endif

namespace hg {

// ------------------------------------------------------------------------------------------------------------------
// f2: two FP32 values processed by one instruction (Blackwell FFMA2/FMUL2/FADD2 on a 64-bit register pair).  The packed
// FP32 path instantiates the whole library with T = f2, the two halves being two helicity configurations of the same
// event that differ in one gluon's helicity: every arithmetic instruction then does the work of two, which halves the
// instruction count of the long straight-line bodies (they are instruction-fetch bound).
// The operators are `mul/add/sub.f32x2` without a rounding modifier, so ptxas contracts a product and a sum into one
// FFMA2 exactly as it does for scalar float (checked in the SASS).  Comparisons look at the first half: they are only
// applied to values that are the same in both halves (chirality signs).
// ------------------------------------------------------------------------------------------------------------------
struct __align__(8) f2 {
    unsigned long long v;             // both halves in one 64-bit register: low word = first configuration, high = second
    f2() = default;
    HG_HD static unsigned int bits(float a) {
#if defined(__CUDA_ARCH__)
        return __float_as_uint(a);
#else
        unsigned int u; memcpy(&u, &a, 4); return u;
#endif
    }
    HG_HD static float val(unsigned int u) {
#if defined(__CUDA_ARCH__)
        return __uint_as_float(u);
#else
        float a; memcpy(&a, &u, 4); return a;
#endif
    }
    HG_HD f2(float a, float b) : v(((unsigned long long)bits(b) << 32) | bits(a)) {}
    HG_HD f2(float a) : f2(a, a) {}
    HG_HD f2(double a) : f2((float)a, (float)a) {}
    HG_HD f2(int a) : f2((float)a, (float)a) {}
    HG_HD float lo() const { return val((unsigned int)v); }
    HG_HD float hi() const { return val((unsigned int)(v >> 32)); }
};
#if defined(__CUDA_ARCH__)
#define HG_F2_BODY(ptx, cexpr) { f2 r; asm(ptx " %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
#else
#define HG_F2_BODY(ptx, cexpr) { return cexpr; }
#endif
HG_HD f2 operator+(f2 a, f2 b) HG_F2_BODY("add.f32x2", f2(a.lo() + b.lo(), a.hi() + b.hi()))
HG_HD f2 operator-(f2 a, f2 b) HG_F2_BODY("sub.f32x2", f2(a.lo() - b.lo(), a.hi() - b.hi()))
HG_HD f2 operator*(f2 a, f2 b) HG_F2_BODY("mul.f32x2", f2(a.lo() * b.lo(), a.hi() * b.hi()))
#undef HG_F2_BODY
HG_HD f2 operator-(f2 a) { f2 r; r.v = a.v ^ 0x8000000080000000ull; return r; }
HG_HD f2& operator+=(f2& a, f2 b) { a = a + b; return a; }
HG_HD f2& operator-=(f2& a, f2 b) { a = a - b; return a; }
HG_HD f2& operator*=(f2& a, f2 b) { a = a * b; return a; }
HG_HD bool operator>(f2 a, f2 b) { return a.lo() > b.lo(); }
HG_HD bool operator<(f2 a, f2 b) { return a.lo() < b.lo(); }
HG_HD bool operator>=(f2 a, f2 b) { return a.lo() >= b.lo(); }
HG_HD bool operator==(f2 a, f2 b) { return a.lo() == b.lo(); }

template <typename T> struct cx { T re, im; };
template <typename T> struct vec4 { cx<T> v[4]; };     // gluon wavefunction / off-shell gluon current
template <typename T> struct mom4 { T p[4]; };         // real 4-momentum
template <typename T> struct sp2 { cx<T> s[2]; };      // Weyl spinor (column psi or row psibar)

template <typename T> HG_HD cx<T> mk(T re, T im) { cx<T> r; r.re = re; r.im = im; return r; }
template <typename T> HG_HD cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <typename T> HG_HD cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <typename T> HG_HD cx<T> operator-(cx<T> a) { return mk<T>(-a.re, -a.im); }
template <typename T> HG_HD cx<T> operator*(cx<T> a, cx<T> b) { return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
template <typename T> HG_HD cx<T> operator*(T s, cx<T> a) { return mk<T>(s * a.re, s * a.im); }
template <typename T> HG_HD cx<T> operator*(cx<T> a, T s) { return mk<T>(s * a.re, s * a.im); }
template <typename T> HG_HD cx<T> conj(cx<T> a) { return mk<T>(a.re, -a.im); }
template <typename T> HG_HD cx<T> times_i(cx<T> a) { return mk<T>(-a.im, a.re); }
template <typename T> HG_HD T norm2(cx<T> a) { return a.re * a.re + a.im * a.im; }

template <typename T> HG_HD mom4<T> operator+(const mom4<T>& a, const mom4<T>& b) { mom4<T> r; for (int m = 0; m < 4; ++m) r.p[m] = a.p[m] + b.p[m]; return r; }
template <typename T> HG_HD mom4<T> operator-(const mom4<T>& a, const mom4<T>& b) { mom4<T> r; for (int m = 0; m < 4; ++m) r.p[m] = a.p[m] - b.p[m]; return r; }
template <typename T> HG_HD mom4<T> operator-(const mom4<T>& a) { mom4<T> r; for (int m = 0; m < 4; ++m) r.p[m] = -a.p[m]; return r; }
template <typename T> HG_HD T mdot(const mom4<T>& a, const mom4<T>& b) { return a.p[0] * b.p[0] - a.p[1] * b.p[1] - a.p[2] * b.p[2] - a.p[3] * b.p[3]; }

// Minkowski products (bilinear, no complex conjugation)
template <typename T> HG_HD cx<T> vdot(const vec4<T>& a, const vec4<T>& b) {
    // one expression per component: every product after the first contracts into an FMA (2 MUL + 14 FMA instead of 8 + 8 + 6 ADD)
    cx<T> r;
    r.re = a.v[0].re * b.v[0].re - a.v[0].im * b.v[0].im - a.v[1].re * b.v[1].re + a.v[1].im * b.v[1].im
         - a.v[2].re * b.v[2].re + a.v[2].im * b.v[2].im - a.v[3].re * b.v[3].re + a.v[3].im * b.v[3].im;
    r.im = a.v[0].re * b.v[0].im + a.v[0].im * b.v[0].re - a.v[1].re * b.v[1].im - a.v[1].im * b.v[1].re
         - a.v[2].re * b.v[2].im - a.v[2].im * b.v[2].re - a.v[3].re * b.v[3].im - a.v[3].im * b.v[3].re;
    return r;
}
template <typename T> HG_HD cx<T> kdot(const mom4<T>& k, const vec4<T>& a) {
    return mk<T>(k.p[0] * a.v[0].re - k.p[1] * a.v[1].re - k.p[2] * a.v[2].re - k.p[3] * a.v[3].re,
                 k.p[0] * a.v[0].im - k.p[1] * a.v[1].im - k.p[2] * a.v[2].im - k.p[3] * a.v[3].im);
}

// ------------------------------------------------------------------------------------------------------------------
// External wavefunctions (step a3).  PAPER.md:219, 471 defer to the paper's ref. [1] and to HELAS (ref. [3]); the
// formulas are the standard massless helicity eigenstates.  Each routine is split into a
// helicity-INDEPENDENT part, evaluated once per event ("*_basis"), and a per-helicity selection that is only a sign.
// ------------------------------------------------------------------------------------------------------------------

// vxxxxx, basis part: for a gluon with physical momentum p fills r[3] = -eps1/sqrt2, i[3] = -+eps2/sqrt2 (spatial parts)
//   eps1 = (px pz, py pz, -pT^2)/(|p| pT),  eps2 = (-py, px, 0)/pT;     on the beam axis eps1 = x^, eps2 = sgn(pz) y^
// so that the helicity-lambda polarisation vector is eps = (0, lambda*r + i*i): (-lambda eps1 - i eps2)/sqrt2 for an
// incoming gluon, its complex conjugate for an outgoing one.
template <typename T> HG_HD void vxxxxx_basis(const T* p, bool initial, T* r, T* i) {
    const T px = p[1], py = p[2], pz = p[3];
    const T pt2 = px * px + py * py;
    const T rs2 = T(0.70710678118654752440);
    const T sg = initial ? -rs2 : rs2;
    if (pt2 == T(0)) {
        r[0] = -rs2; r[1] = T(0); r[2] = T(0);
        i[0] = T(0); i[1] = (pz >= T(0)) ? sg : -sg; i[2] = T(0);
    } else {
        const T pp = sqrt(pt2 + pz * pz), pt = sqrt(pt2);
        const T a = -rs2 / (pp * pt), b = sg / pt;
        r[0] = a * px * pz; r[1] = a * py * pz; r[2] = -a * pt2;
        i[0] = -b * py; i[1] = b * px; i[2] = T(0);
    }
}
// vxxxxx, helicity part: lambda = +-1
template <typename T> HG_HD vec4<T> vxxxxx(const T* r, const T* i, T lambda) {
    vec4<T> w;
    w.v[0] = mk<T>(T(0), T(0));
    w.v[1] = mk<T>(lambda * r[0], i[0]); w.v[2] = mk<T>(lambda * r[1], i[1]); w.v[3] = mk<T>(lambda * r[2], i[2]);
    return w;
}

// ixxxxx / oxxxxx, basis part: the two massless Weyl spinors of physical momentum p from 3 reals s = (w, ax, ay),
//   w = sqrt(E + pz), (ax, ay) = (px, py)/w:    phi_L = (-ax + i ay, w)   [solves (p.sigmabar) phi = 0, chi = +1]
//                                               phi_R = (w, ax + i ay)    [solves (p.sigma) phi = 0,    chi = -1]
// E + pz is formed without cancellation (pT^2/(E - pz) when pz < 0); on the -z axis the limit w = 0, (ax, ay) = (sqrt(2E), 0)
// is taken (reading A19: any finite normalised choice, phases are free).
template <typename T> HG_HD void ixxxxx_basis(const T* p, T* s) {
    const T e = p[0], px = p[1], py = p[2], pz = p[3];
    const T pt2 = px * px + py * py;
    if (pt2 == T(0) && pz < T(0)) { s[0] = T(0); s[1] = sqrt(e + e); s[2] = T(0); return; }
    const T epz = (pz >= T(0)) ? (e + pz) : pt2 / (e - pz);
    const T w = sqrt(epz), iw = T(1) / w;
    s[0] = w; s[1] = px * iw; s[2] = py * iw;
}
// flowing-in (column) spinor of a line with chirality chi
template <typename T> HG_HD sp2<T> ixxxxx(const T* s, T chi) {
    sp2<T> f;
    if (chi > T(0)) { f.s[0] = mk<T>(-s[1], s[2]); f.s[1] = mk<T>(s[0], T(0)); }
    else            { f.s[0] = mk<T>(s[0], T(0));  f.s[1] = mk<T>(s[1], s[2]); }
    return f;
}
// flowing-out (row) spinor: the Dirac conjugate, whose non-zero half is the complex conjugate of the column spinor
template <typename T> HG_HD sp2<T> oxxxxx(const T* s, T chi) {
    sp2<T> f = ixxxxx<T>(s, chi);
    f.s[0].im = -f.s[0].im; f.s[1].im = -f.s[1].im;
    return f;
}

// ------------------------------------------------------------------------------------------------------------------
// Three-gluon vertex (section 4.1).  V3(a,ka; b,kb; c,kc), all momenta into the vertex:
//   V3 = (a.b)((ka-kb).c) + (b.c)((kb-kc).a) + (c.a)((kc-ka).b)
// ------------------------------------------------------------------------------------------------------------------

// vvvxxx: amplitude of the ggg vertex from three (on- or off-shell) gluon wavefunctions; colour factor i f^{abc}
// (eq. 27).  Arguments as eq. 24 plus the momenta flowing INTO the vertex.
template <typename T> HG_VX cx<T> vvvxxx(HG_CV4 ga, HG_CM4 ka, HG_CV4 gb, HG_CM4 kb,
                                         HG_CV4 gc, HG_CM4 kc, T g) {
    const cx<T> ab = vdot(ga, gb), bc = vdot(gb, gc), ca = vdot(gc, ga);
    const cx<T> v = ab * kdot(ka - kb, gc) + bc * kdot(kb - kc, ga) + ca * kdot(kc - ka, gb);
    return g * v;
}

// jvvxx0: off-shell gluon current j^mu(gc: ga, gb) from the ggg vertex with the Feynman-gauge propagator (section 4.1.2,
// PAPER.md:292-313; surviving fragments of List 2); colour factor i f^{abc} (eq. 30).
// q = -(ka + kb) is the momentum of the third leg flowing into the vertex; inv_q2 = 1/q^2.
//   j^mu = g/q^2 [ (a.b)(ka-kb)^mu + b^mu ((kb-q).a) + a^mu ((q-ka).b) ],  kb - q = ka + 2 kb,  q - ka = -(2 ka + kb)
template <typename T> HG_VX vec4<T> jvvxx0(HG_CV4 ga, HG_CM4 ka, HG_CV4 gb, HG_CM4 kb, T g, T inv_q2) {
    const T gs = g * inv_q2;
    const cx<T> ab = gs * vdot(ga, gb);
    const cx<T> sa = gs * kdot(ka + kb + kb, ga);
    const cx<T> sb = -(gs * kdot(ka + ka + kb, gb));
    vec4<T> j;
    for (int m = 0; m < 4; ++m) j.v[m] = ab * (ka.p[m] - kb.p[m]) + sa * gb.v[m] + sb * ga.v[m];
    return j;
}

// ------------------------------------------------------------------------------------------------------------------
// Four-gluon vertex (section 4.2).  The vertex of eq. 31 is the sum of three colour structures
// (eq. 36), each multiplying -g^2 W_piece:
//   piece 0, f^{abe}f^{cde}:  W0 = (a.c)(b.d) - (a.d)(b.c)      ("the first and the third, and hence also the second and
//   piece 1, f^{ace}f^{dbe}:  W1 = (a.d)(c.b) - (a.b)(c.d)        the fourth gluon wave functions are contracted")
//   piece 2, f^{ade}f^{bce}:  W2 = (a.b)(d.c) - (a.c)(d.b)
// W1 and W2 are W0 with the arguments permuted as in eqs. 35b, 35c: (a,c,d,b) and (a,d,b,c).
// ------------------------------------------------------------------------------------------------------------------

// ggggxx: one colour-structure piece of the gggg amplitude (call three times with permuted arguments, eq. 35)
template <typename T> HG_HD cx<T> ggggxx(const vec4<T>& ga, const vec4<T>& gb, const vec4<T>& gc, const vec4<T>& gd, T gg) {
    return gg * (vdot(ga, gd) * vdot(gb, gc) - vdot(ga, gc) * vdot(gb, gd));
}
// the three pieces at once (the six pair products are shared): v[0..2] for f^{abe}f^{cde}, f^{ace}f^{dbe}, f^{ade}f^{bce}
template <typename T> HG_HD void ggggxx3(const vec4<T>& ga, const vec4<T>& gb, const vec4<T>& gc, const vec4<T>& gd, T gg, cx<T>* v) {
    const cx<T> x = vdot(ga, gb) * vdot(gc, gd), y = vdot(ga, gc) * vdot(gb, gd), z = vdot(ga, gd) * vdot(gb, gc);
    v[0] = gg * (z - y); v[1] = gg * (x - z); v[2] = gg * (y - x);
}

// jgggx0: off-shell gluon current from the gggg vertex, one colour-structure piece (section 4.2.2),
// Feynman-gauge propagator 1/q^2 of the fourth leg:  j^mu = d ggggxx(ga,gb,gc,gd) / d gd_mu / q^2
//   = gg/q^2 [ (b.c) a^mu - (a.c) b^mu ]          (mirror identity ggggxx(a,b,c,d) = q^2 (jgggx0(a,b,c) . d), reading A6)
template <typename T> HG_HD vec4<T> jgggx0(const vec4<T>& ga, const vec4<T>& gb, const vec4<T>& gc, T gg, T inv_q2) {
    const T s = gg * inv_q2;
    const cx<T> bc = s * vdot(gb, gc), ac = s * vdot(ga, gc);
    vec4<T> j;
    for (int m = 0; m < 4; ++m) j.v[m] = bc * ga.v[m] - ac * gb.v[m];
    return j;
}
// the three pieces at once: j[0] = jgggx0(a,b,c), j[1] = jgggx0(a,c,d->b) ... in the open-leg form of eq. 40
//   j0 = (b.c) a - (a.c) b,   j1 = (a.b) c - (b.c) a,   j2 = (a.c) b - (a.b) c      (times gg/q^2)
template <typename T> HG_HD void jgggx03(const vec4<T>& ga, const vec4<T>& gb, const vec4<T>& gc, T gg, T inv_q2, vec4<T>* j) {
    const T s = gg * inv_q2;
    const cx<T> ab = s * vdot(ga, gb), ac = s * vdot(ga, gc), bc = s * vdot(gb, gc);
    for (int m = 0; m < 4; ++m) {
        const cx<T> A = bc * ga.v[m], B = ac * gb.v[m], C = ab * gc.v[m];
        j[0].v[m] = A - B; j[1].v[m] = C - A; j[2].v[m] = B - C;
    }
}

// piece-indexed forms used by the generated code: piece 0, 1, 2 = the argument permutations of eqs. 35a-c
template <typename T> HG_VX cx<T> ggggxxp(HG_CV4 ga, HG_CV4 gb, HG_CV4 gc, HG_CV4 gd, int piece) {
    if (piece == 0) return ggggxx<T>(ga, gb, gc, gd, T(1));
    if (piece == 1) return ggggxx<T>(ga, gc, gd, gb, T(1));
    return ggggxx<T>(ga, gd, gb, gc, T(1));
}
template <typename T> HG_VX vec4<T> jgggx0p(HG_CV4 ga, HG_CV4 gb, HG_CV4 gc, int piece, T inv_q2) {
    if (piece == 0) return jgggx0<T>(ga, gb, gc, T(1), inv_q2);      // (b.c) a - (a.c) b
    if (piece == 1) return jgggx0<T>(gc, ga, gb, T(1), inv_q2);      // (a.b) c - (c.b) a
    return jgggx0<T>(gb, gc, ga, T(1), inv_q2);                      // (c.a) b - (b.a) c
}

// ------------------------------------------------------------------------------------------------------------------
// Quark-gluon vertex (eqs. 18-22): identical to the qq-photon functions of the paper's ref. [1] except
// for the coupling; colour factor -T^a per vertex (eq. 22).  Chiral representation gamma^mu = [[0, sigma^mu],[sigmabar^mu, 0]];
// a massless line of chirality chi only ever populates one 2-component half, and
//   slash(v) acts on it as the 2x2 matrix  S(v; s) = v0 + s (v . sigma) = [[v0 + s v3, s (v1 - i v2)], [s (v1 + i v2), v0 - s v3]]
// with s = +chi where a polarisation vector sits and s = -chi where the propagator momentum sits.
// ------------------------------------------------------------------------------------------------------------------
template <typename T> HG_HD sp2<T> smul_col(const vec4<T>& v, T s, const sp2<T>& f) {       // S(v; s) f
    const cx<T> d0 = v.v[0] + s * v.v[3], d1 = v.v[0] - s * v.v[3];
    const cx<T> om = s * (v.v[1] - times_i(v.v[2])), op = s * (v.v[1] + times_i(v.v[2]));
    sp2<T> r; r.s[0] = d0 * f.s[0] + om * f.s[1]; r.s[1] = op * f.s[0] + d1 * f.s[1]; return r;
}
template <typename T> HG_HD sp2<T> smul_row(const sp2<T>& f, const vec4<T>& v, T s) {       // f S(v; s)
    const cx<T> d0 = v.v[0] + s * v.v[3], d1 = v.v[0] - s * v.v[3];
    const cx<T> om = s * (v.v[1] - times_i(v.v[2])), op = s * (v.v[1] + times_i(v.v[2]));
    sp2<T> r; r.s[0] = f.s[0] * d0 + f.s[1] * op; r.s[1] = f.s[0] * om + f.s[1] * d1; return r;
}
template <typename T> HG_HD sp2<T> kmul_col(const mom4<T>& k, T s, const sp2<T>& f, T c) {  // c S(k; s) f, k real
    const T d0 = c * (k.p[0] + s * k.p[3]), d1 = c * (k.p[0] - s * k.p[3]), ox = c * s * k.p[1], oy = c * s * k.p[2];
    sp2<T> r;   // (ox - i oy) f1 ; (ox + i oy) f0
    r.s[0] = mk<T>(d0 * f.s[0].re + ox * f.s[1].re + oy * f.s[1].im, d0 * f.s[0].im + ox * f.s[1].im - oy * f.s[1].re);
    r.s[1] = mk<T>(d1 * f.s[1].re + ox * f.s[0].re - oy * f.s[0].im, d1 * f.s[1].im + ox * f.s[0].im + oy * f.s[0].re);
    return r;
}
template <typename T> HG_HD sp2<T> kmul_row(const sp2<T>& f, const mom4<T>& k, T s, T c) {  // c f S(k; s), k real
    const T d0 = c * (k.p[0] + s * k.p[3]), d1 = c * (k.p[0] - s * k.p[3]), ox = c * s * k.p[1], oy = c * s * k.p[2];
    sp2<T> r;   // r0 = f0 d0 + f1 (ox + i oy) ; r1 = f0 (ox - i oy) + f1 d1
    r.s[0] = mk<T>(d0 * f.s[0].re + ox * f.s[1].re - oy * f.s[1].im, d0 * f.s[0].im + ox * f.s[1].im + oy * f.s[1].re);
    r.s[1] = mk<T>(d1 * f.s[1].re + ox * f.s[0].re + oy * f.s[0].im, d1 * f.s[1].im + ox * f.s[0].im - oy * f.s[0].re);
    return r;
}

// iovxx0: amplitude of the qqg vertex (eq. 20; g[0] = g[1] = g, eq. 21):  g fo S(vc; chi) fi
template <typename T> HG_VX cx<T> iovxx0(HG_CS2 fi, HG_CS2 fo, HG_CV4 vc, T chi, T g) {
    const sp2<T> t = smul_col(vc, chi, fi);
    return g * (fo.s[0] * t.s[0] + fo.s[1] * t.s[1]);
}
// fvixx0: off-shell flowing-in quark from a flowing-in quark and a gluon, massless propagator.
// k = momentum of the new line along the fermion arrow (= sum of the incoming momenta behind it); inv_k2 = 1/k^2.
//   fvi = -g/k^2  S(k; -chi) S(vc; chi) fi
template <typename T> HG_VX sp2<T> fvixx0(HG_CS2 fi, HG_CV4 vc, HG_CM4 k, T chi, T g, T inv_k2) {
    return kmul_col(k, -chi, smul_col(vc, chi, fi), -g * inv_k2);
}
// fvoxx0: off-shell flowing-out quark from a flowing-out quark and a gluon.  Here the arrow points from the root towards
// the leaves, so the momentum along it is MINUS the sum of the incoming momenta behind the line: pass that sum as ksum.
//   fvo = -g/k^2  fo S(vc; chi) S(-ksum; -chi)
template <typename T> HG_VX sp2<T> fvoxx0(HG_CS2 fo, HG_CV4 vc, HG_CM4 ksum, T chi, T g, T inv_k2) {
    return kmul_row(smul_row(fo, vc, chi), ksum, -chi, g * inv_k2);
}
// jioxx0: off-shell gluon from a quark pair, Feynman-gauge propagator:  j^mu = g/q^2 fo sigma_chi^mu fi,
// sigma_chi^mu = (1, -chi sigma^i)
template <typename T> HG_VX vec4<T> jioxx0(HG_CS2 fi, HG_CS2 fo, T chi, T g, T inv_q2) {
    const T c = g * inv_q2, cs = -chi * c;
    const cx<T> a00 = fo.s[0] * fi.s[0], a11 = fo.s[1] * fi.s[1], a01 = fo.s[0] * fi.s[1], a10 = fo.s[1] * fi.s[0];
    vec4<T> j;
    j.v[0] = c * (a00 + a11);
    j.v[1] = cs * (a01 + a10);
    j.v[2] = cs * times_i(a10 - a01);
    j.v[3] = cs * (a00 - a11);
    return j;
}

}  // namespace hg
