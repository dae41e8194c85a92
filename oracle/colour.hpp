// ORACLE (test infrastructure only).
//
// Colour by brute force: every colour object is a dense array over ALL colour assignments
// {c_i} of the external legs (1..3 for quark legs, 1..8 for gluons), built by
// contracting the numeric T^a_{ij} and f^{abc} of su3.hpp along the diagram.
//   * colour basis T_alpha^{c_i}                                     (eq. 8,  PAPER.md:81-83)
//   * colour matrix  C_{alpha beta} = sum_{c_i} T_alpha (T_beta)^*   (eq. 9 without 1/(n_a n_b); reading A16)
//   * coefficients of diagram l on the basis, D_l^{c} = sum_alpha coef_{alpha l} T_alpha^{c}, obtained
//     NUMERICALLY: b_beta = sum_c (T_beta^c)^* D_l^c, solve C coef = b by pseudo-inverse, and verify that
//     the residual vanishes on every assignment                       (SURVEY.md 8(c) tier O2)
//
// Bases (reading A12, Table 1):
//   no quark line : Tr(T^{a_0} T^{a_s(1)} ... T^{a_s(n-1)}),  (n-1)! permutations            (eq. 17)
//   one quark line: (T^{a_s(1)} ... T^{a_s(k)})_{i j}, i = colour of the out-end, j of the in-end,  k!
//   two quark lines: for every pairing and every ordered split of a permutation of the k gluons into four
//     lists (A,B,C,D):  sum_e (T^A T^e T^B)_{i1 j1} (T^C T^e T^D)_{i2 j2},  #pairings * k! * C(k+3,3)
//     (an over-complete set; only J^dagger C J is unique, A13).
#pragma once
#include <vector>
#include <cstdint>
#include <cstring>
#include <algorithm>
#include "su3.hpp"
#include "diagrams.hpp"

namespace orc {

struct CTensor {                 // v[compact(legs) * rdim + r]; first leg slowest
    std::vector<int> legs, dims;
    int rdim;
    std::vector<cplx> v;
    size_t n_compact() const { size_t n = 1; for (size_t i = 0; i < dims.size(); ++i) n *= dims[i]; return n; }
};

struct SparseVec { std::vector<uint32_t> idx; std::vector<cplx> val; };

inline int leg_dim(const Process& P, int leg) { return P.legs[leg].kind == LEG_G ? 8 : 3; }
inline int ptype_dim(int ptype) { return ptype == PT_G ? 8 : 3; }

// offsets of the compact indices of `sub` inside the compact index space of `merged`
inline std::vector<size_t> embed_offsets(const CTensor& sub, const std::vector<int>& merged_legs, const std::vector<int>& merged_dims) {
    std::vector<size_t> stride_m(merged_legs.size());
    size_t s = 1;
    for (int i = (int)merged_legs.size() - 1; i >= 0; --i) { stride_m[i] = s; s *= merged_dims[i]; }
    std::vector<size_t> stride_of_sub(sub.legs.size());
    for (size_t i = 0; i < sub.legs.size(); ++i) {
        size_t pos = std::find(merged_legs.begin(), merged_legs.end(), sub.legs[i]) - merged_legs.begin();
        stride_of_sub[i] = stride_m[pos];
    }
    const size_t n = sub.n_compact();
    std::vector<size_t> off(n);
    for (size_t c = 0; c < n; ++c) {
        size_t rem = c, o = 0;
        for (int i = (int)sub.legs.size() - 1; i >= 0; --i) { o += (rem % sub.dims[i]) * stride_of_sub[i]; rem /= sub.dims[i]; }
        off[c] = o;
    }
    return off;
}

// colour tensor of the subtree below node `id` (recursive, literal contraction)
inline CTensor node_colour(const DiagramSet& D, int id) {
    const SU3& G = su3();
    const Node& n = D.nodes[id];
    CTensor out;
    out.rdim = ptype_dim(n.ptype);
    if (n.kind == NK_LEAF) {
        out.legs.push_back(n.leg); out.dims.push_back(out.rdim);
        out.v.assign((size_t)out.rdim * out.rdim, 0.0);
        for (int c = 0; c < out.rdim; ++c) out.v[(size_t)c * out.rdim + c] = 1.0;
        return out;
    }
    const int nch = (n.kind == NK_GGGG) ? 3 : 2;
    CTensor ch[3];
    for (int i = 0; i < nch; ++i) ch[i] = node_colour(D, n.ch[i]);
    for (int i = 0; i < nch; ++i) out.legs.insert(out.legs.end(), ch[i].legs.begin(), ch[i].legs.end());
    std::sort(out.legs.begin(), out.legs.end());
    for (size_t i = 0; i < out.legs.size(); ++i) out.dims.push_back(leg_dim(D.proc, out.legs[i]));
    out.v.assign(out.n_compact() * out.rdim, 0.0);
    std::vector<size_t> off[3];
    for (int i = 0; i < nch; ++i) off[i] = embed_offsets(ch[i], out.legs, out.dims);

    if (nch == 2) {
        const int ra = ch[0].rdim, rb = ch[1].rdim, rc = out.rdim;
        // coupling K[a][b][c]
        std::vector<cplx> K((size_t)ra * rb * rc, 0.0);
        for (int a = 0; a < ra; ++a) for (int b = 0; b < rb; ++b) for (int c = 0; c < rc; ++c) {
            cplx k = 0.0;
            if (n.kind == NK_GGG)        k = G.f[a][b][c];        // f^{abc}: (child0, child1, parent)
            else if (n.kind == NK_QQG_G) k = G.T[c][a][b];        // T^c_{ij}: i = psibar child, j = psi child
            else if (n.kind == NK_QG_Q)  k = G.T[b][c][a];        // T^b_{ij}: i = parent, j = psi child
            else if (n.kind == NK_BG_B)  k = G.T[b][a][c];        // T^b_{ij}: i = psibar child, j = parent
            K[((size_t)a * rb + b) * rc + c] = k;
        }
        const size_t na = ch[0].n_compact(), nb = ch[1].n_compact();
        for (size_t ia = 0; ia < na; ++ia) for (int a = 0; a < ra; ++a) {
            const cplx va = ch[0].v[ia * ra + a];
            if (va == 0.0) continue;
            for (size_t ib = 0; ib < nb; ++ib) for (int b = 0; b < rb; ++b) {
                const cplx vb = ch[1].v[ib * rb + b];
                if (vb == 0.0) continue;
                cplx* o = &out.v[(off[0][ia] + off[1][ib]) * rc];
                const cplx* k = &K[((size_t)a * rb + b) * rc];
                for (int c = 0; c < rc; ++c) o[c] += va * vb * k[c];
            }
        }
    } else {
        // gggg colour structures of eq. 36, legs (a,b,c,d) = (child0, child1, child2, parent)
        std::vector<double> K4(8 * 8 * 8 * 8, 0.0);
        for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) for (int d = 0; d < 8; ++d) {
            double k = 0.0;
            for (int e = 0; e < 8; ++e) {
                if (n.piece == 0)      k += G.f[a][b][e] * G.f[c][d][e];
                else if (n.piece == 1) k += G.f[a][c][e] * G.f[b][d][e];
                else                   k += G.f[a][d][e] * G.f[b][c][e];
            }
            K4[((a * 8 + b) * 8 + c) * 8 + d] = k;
        }
        const size_t na = ch[0].n_compact(), nb = ch[1].n_compact(), nc = ch[2].n_compact();
        for (size_t ia = 0; ia < na; ++ia) for (int a = 0; a < 8; ++a) {
            const cplx va = ch[0].v[ia * 8 + a]; if (va == 0.0) continue;
            for (size_t ib = 0; ib < nb; ++ib) for (int b = 0; b < 8; ++b) {
                const cplx vb = ch[1].v[ib * 8 + b]; if (vb == 0.0) continue;
                for (size_t ic = 0; ic < nc; ++ic) for (int c = 0; c < 8; ++c) {
                    const cplx vc = ch[2].v[ic * 8 + c]; if (vc == 0.0) continue;
                    cplx* o = &out.v[(off[0][ia] + off[1][ib] + off[2][ic]) * 8];
                    const double* k = &K4[((a * 8 + b) * 8 + c) * 8];
                    for (int d = 0; d < 8; ++d) o[d] += va * vb * vc * k[d];
                }
            }
        }
    }
    return out;
}

// ---- colour basis -----------------------------------------------------------------------
struct BasisElement {
    int kind;                     // 0 trace, 1 one string, 2 two strings joined by a gluon
    int pairing;
    std::vector<int> seq[4];      // kind 0: seq[0] = trace order; kind 1: seq[0] = string; kind 2: A,B,C,D
};

inline void mat_identity(cplx M[3][3]) { for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) M[i][j] = (i == j) ? 1.0 : 0.0; }
inline void mat_mul_T(cplx M[3][3], int a) {         // M <- M T^a
    const SU3& G = su3();
    cplx R[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { cplx s = 0.0; for (int k = 0; k < 3; ++k) s += M[i][k] * G.T[a][k][j]; R[i][j] = s; }
    std::memcpy(M, R, sizeof(R));
}

inline std::vector<BasisElement> build_basis(const DiagramSet& D) {
    const Process& P = D.proc;
    std::vector<int> gl;
    for (int i = 0; i < P.n_ext(); ++i) if (P.legs[i].kind == LEG_G) gl.push_back(i);
    const size_t n_lines = D.pairings[0].in_leg.size();
    std::vector<BasisElement> B;
    if (n_lines == 0) {
        std::vector<int> rest(gl.begin() + 1, gl.end());
        do {
            BasisElement e; e.kind = 0; e.pairing = 0;
            e.seq[0].push_back(gl[0]); e.seq[0].insert(e.seq[0].end(), rest.begin(), rest.end());
            B.push_back(e);
        } while (std::next_permutation(rest.begin(), rest.end()));
    } else if (n_lines == 1) {
        std::vector<int> perm = gl;
        do { BasisElement e; e.kind = 1; e.pairing = 0; e.seq[0] = perm; B.push_back(e); }
        while (std::next_permutation(perm.begin(), perm.end()));
    } else if (n_lines == 2) {
        const int k = (int)gl.size();
        for (size_t ip = 0; ip < D.pairings.size(); ++ip) {
            std::vector<int> perm = gl;
            do {
                for (int c1 = 0; c1 <= k; ++c1) for (int c2 = c1; c2 <= k; ++c2) for (int c3 = c2; c3 <= k; ++c3) {
                    BasisElement e; e.kind = 2; e.pairing = (int)ip;
                    e.seq[0].assign(perm.begin(), perm.begin() + c1);
                    e.seq[1].assign(perm.begin() + c1, perm.begin() + c2);
                    e.seq[2].assign(perm.begin() + c2, perm.begin() + c3);
                    e.seq[3].assign(perm.begin() + c3, perm.end());
                    B.push_back(e);
                }
            } while (std::next_permutation(perm.begin(), perm.end()));
        }
    } else throw std::runtime_error("oracle colour basis: at most two quark lines");
    return B;
}

// value of a basis element on one colour assignment col[leg]
inline cplx basis_value(const DiagramSet& D, const BasisElement& e, const int* col) {
    const SU3& G = su3();
    if (e.kind == 0) {
        cplx M[3][3]; mat_identity(M);
        for (size_t i = 0; i < e.seq[0].size(); ++i) mat_mul_T(M, col[e.seq[0][i]]);
        return M[0][0] + M[1][1] + M[2][2];
    }
    const Pairing& pr = D.pairings[e.pairing];
    if (e.kind == 1) {
        cplx M[3][3]; mat_identity(M);
        for (size_t i = 0; i < e.seq[0].size(); ++i) mat_mul_T(M, col[e.seq[0][i]]);
        return M[col[pr.out_leg[0]]][col[pr.in_leg[0]]];
    }
    cplx r = 0.0;
    for (int x = 0; x < 8; ++x) {
        cplx M1[3][3], M2[3][3]; mat_identity(M1); mat_identity(M2);
        for (size_t i = 0; i < e.seq[0].size(); ++i) mat_mul_T(M1, col[e.seq[0][i]]);
        mat_mul_T(M1, x);
        for (size_t i = 0; i < e.seq[1].size(); ++i) mat_mul_T(M1, col[e.seq[1][i]]);
        for (size_t i = 0; i < e.seq[2].size(); ++i) mat_mul_T(M2, col[e.seq[2][i]]);
        mat_mul_T(M2, x);
        for (size_t i = 0; i < e.seq[3].size(); ++i) mat_mul_T(M2, col[e.seq[3][i]]);
        r += M1[col[pr.out_leg[0]]][col[pr.in_leg[0]]] * M2[col[pr.out_leg[1]]][col[pr.in_leg[1]]];
    }
    (void)G;
    return r;
}

// symmetric eigen-decomposition by cyclic Jacobi rotations (plain textbook routine)
inline void jacobi_eigen(int n, std::vector<double> A, std::vector<double>& eval, std::vector<double>& evec) {
    evec.assign((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) evec[(size_t)i * n + i] = 1.0;
    for (int sweep = 0; sweep < 100; ++sweep) {
        double offd = 0.0;
        for (int p = 0; p < n; ++p) for (int q = p + 1; q < n; ++q) offd += A[(size_t)p * n + q] * A[(size_t)p * n + q];
        if (offd < 1e-28) break;
        for (int p = 0; p < n; ++p) for (int q = p + 1; q < n; ++q) {
            const double apq = A[(size_t)p * n + q];
            if (std::fabs(apq) < 1e-300) continue;
            const double theta = (A[(size_t)q * n + q] - A[(size_t)p * n + p]) / (2.0 * apq);
            const double t = ((theta >= 0.0) ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
            const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
            for (int k = 0; k < n; ++k) {
                const double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
                A[(size_t)k * n + p] = c * akp - s * akq; A[(size_t)k * n + q] = s * akp + c * akq;
            }
            for (int k = 0; k < n; ++k) {
                const double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
                A[(size_t)p * n + k] = c * apk - s * aqk; A[(size_t)q * n + k] = s * apk + c * aqk;
            }
            for (int k = 0; k < n; ++k) {
                const double vkp = evec[(size_t)k * n + p], vkq = evec[(size_t)k * n + q];
                evec[(size_t)k * n + p] = c * vkp - s * vkq; evec[(size_t)k * n + q] = s * vkp + c * vkq;
            }
        }
    }
    eval.resize(n);
    for (int i = 0; i < n; ++i) eval[i] = A[(size_t)i * n + i];
}

struct ColourData {
    int m;                                  // number of basis elements
    size_t n_assign;                        // number of colour assignments
    std::vector<BasisElement> basis;
    std::vector<SparseVec> basis_val;       // T_alpha^{c}, sparse over assignments
    std::vector<double> C;                  // m x m, real symmetric
    double C_max_imag, C_max_asym;
    std::vector<double> eval, evec;         // of C
    int rank;
    // coefficient table coef[l] = sparse list of (alpha, coefficient) with D_l = sum coef T_alpha
    std::vector<std::vector<std::pair<int, cplx> > > coef;
    double max_residual;                    // max over diagrams and assignments of |D_l - sum coef T_alpha|
    std::vector<SparseVec> diag_colour;     // D_l^{c} (kept only on request, for tier O1)
    double frac_nonzero_pairs, frac_all_zero;   // Monte-Carlo colour statistics
};

inline void build_colour(const DiagramSet& D, ColourData& cd, bool keep_diagram_colour) {
    const Process& P = D.proc;
    const int n = P.n_ext();
    std::vector<int> dims(n);
    size_t N = 1;
    for (int i = 0; i < n; ++i) { dims[i] = leg_dim(P, i); N *= dims[i]; }
    cd.n_assign = N;
    cd.basis = build_basis(D);
    cd.m = (int)cd.basis.size();
    const int m = cd.m;
    cd.basis_val.assign(m, SparseVec());
    #pragma omp parallel for schedule(dynamic)
    for (int al = 0; al < m; ++al) {
        std::vector<int> col(n);
        for (size_t c = 0; c < N; ++c) {
            size_t rem = c;
            for (int i = n - 1; i >= 0; --i) { col[i] = (int)(rem % dims[i]); rem /= dims[i]; }
            const cplx v = basis_value(D, cd.basis[al], col.data());
            if (std::abs(v) > 1e-14) { cd.basis_val[al].idx.push_back((uint32_t)c); cd.basis_val[al].val.push_back(v); }
        }
    }
    // Monte-Carlo colour statistics
    {
        std::vector<char> any(N, 0);
        size_t nz = 0;
        for (int al = 0; al < m; ++al) { nz += cd.basis_val[al].idx.size(); for (size_t k = 0; k < cd.basis_val[al].idx.size(); ++k) any[cd.basis_val[al].idx[k]] = 1; }
        size_t nany = 0; for (size_t c = 0; c < N; ++c) nany += any[c];
        cd.frac_nonzero_pairs = (double)nz / ((double)N * m);
        cd.frac_all_zero = 1.0 - (double)nany / (double)N;
    }
    // colour matrix, eq. 9 without the 1/(n_a n_b)
    cd.C.assign((size_t)m * m, 0.0);
    std::vector<double> Cim((size_t)m * m, 0.0);
    #pragma omp parallel for schedule(dynamic)
    for (int al = 0; al < m; ++al) {
        std::vector<cplx> dense(N, 0.0);
        for (size_t k = 0; k < cd.basis_val[al].idx.size(); ++k) dense[cd.basis_val[al].idx[k]] = cd.basis_val[al].val[k];
        for (int be = 0; be < m; ++be) {
            cplx s = 0.0;
            const SparseVec& tb = cd.basis_val[be];
            for (size_t k = 0; k < tb.idx.size(); ++k) s += dense[tb.idx[k]] * std::conj(tb.val[k]);
            cd.C[(size_t)al * m + be] = s.real(); Cim[(size_t)al * m + be] = s.imag();
        }
    }
    cd.C_max_imag = 0.0; cd.C_max_asym = 0.0;
    for (int a = 0; a < m; ++a) for (int b = 0; b < m; ++b) {
        cd.C_max_imag = std::max(cd.C_max_imag, std::fabs(Cim[(size_t)a * m + b]));
        cd.C_max_asym = std::max(cd.C_max_asym, std::fabs(cd.C[(size_t)a * m + b] - cd.C[(size_t)b * m + a]));
    }
    jacobi_eigen(m, cd.C, cd.eval, cd.evec);
    double emax = 0.0; for (int i = 0; i < m; ++i) emax = std::max(emax, std::fabs(cd.eval[i]));
    cd.rank = 0; for (int i = 0; i < m; ++i) if (cd.eval[i] > 1e-9 * emax) cd.rank += 1;

    // diagram colour tensors and their coefficients on the basis
    const int nd = (int)D.diagrams.size();
    cd.coef.assign(nd, std::vector<std::pair<int, cplx> >());
    if (keep_diagram_colour) cd.diag_colour.assign(nd, SparseVec());
    double max_res = 0.0;
    #pragma omp parallel for schedule(dynamic) reduction(max : max_res)
    for (int l = 0; l < nd; ++l) {
        CTensor t = node_colour(D, D.diagrams[l]);      // legs = all but the root (the last leg), root index fastest
        std::vector<cplx>& Dl = t.v;                    // == D_l over all assignments, first leg slowest
        std::vector<cplx> b(m);
        for (int be = 0; be < m; ++be) {
            cplx s = 0.0;
            const SparseVec& tb = cd.basis_val[be];
            for (size_t k = 0; k < tb.idx.size(); ++k) s += std::conj(tb.val[k]) * Dl[tb.idx[k]];
            b[be] = s;
        }
        // pseudo-inverse: coef = sum_k v_k (v_k . b) / lambda_k over non-null eigenvalues
        std::vector<cplx> x(m, 0.0);
        for (int k = 0; k < m; ++k) {
            if (!(cd.eval[k] > 1e-9 * emax)) continue;
            cplx vb = 0.0;
            for (int i = 0; i < m; ++i) vb += cd.evec[(size_t)i * m + k] * b[i];
            for (int i = 0; i < m; ++i) x[i] += cd.evec[(size_t)i * m + k] * vb / cd.eval[k];
        }
        if (keep_diagram_colour)
            for (size_t c = 0; c < N; ++c) if (std::abs(Dl[c]) > 1e-14) { cd.diag_colour[l].idx.push_back((uint32_t)c); cd.diag_colour[l].val.push_back(Dl[c]); }
        for (int al = 0; al < m; ++al) {
            if (std::abs(x[al]) < 1e-11) continue;
            cd.coef[l].push_back(std::make_pair(al, x[al]));
            const SparseVec& ta = cd.basis_val[al];
            for (size_t k = 0; k < ta.idx.size(); ++k) Dl[ta.idx[k]] -= x[al] * ta.val[k];
        }
        double res = 0.0;
        for (size_t c = 0; c < N; ++c) res = std::max(res, std::abs(Dl[c]));
        max_res = std::max(max_res, res);
    }
    cd.max_residual = max_res;
}
}  // namespace orc
