// ORACLE (test infrastructure only -- never linked, imported or called by the product path).
//
// SU(3) tables for the brute-force colour sums of the oracle.
// PAPER.md:83  "color bases T_alpha^{c_i} which are made from the SU(3) generators in the
//               fundamental representation"; P:79 colour indices 1..3 (quarks), 1..8 (gluons).
// Normalisation used throughout: T^a = lambda^a / 2, Tr(T^a T^b) = delta^{ab}/2,
// [T^a, T^b] = i f^{abc} T^c.  The structure constants are NOT typed in: they are computed
// from the commutator definition,  f^{abc} = -2i Tr([T^a,T^b] T^c).
#pragma once
#include <complex>
#include <cmath>

namespace orc {
typedef std::complex<double> cplx;

struct SU3 {
    cplx T[8][3][3];      // T^a_{ij}
    double f[8][8][8];    // f^{abc}
    SU3() {
        const cplx I(0.0, 1.0);
        cplx L[8][3][3];
        for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) L[a][i][j] = 0.0;
        // Gell-Mann matrices lambda^1 .. lambda^8
        L[0][0][1] = 1.0;  L[0][1][0] = 1.0;
        L[1][0][1] = -I;   L[1][1][0] = I;
        L[2][0][0] = 1.0;  L[2][1][1] = -1.0;
        L[3][0][2] = 1.0;  L[3][2][0] = 1.0;
        L[4][0][2] = -I;   L[4][2][0] = I;
        L[5][1][2] = 1.0;  L[5][2][1] = 1.0;
        L[6][1][2] = -I;   L[6][2][1] = I;
        const double s3 = 1.0 / std::sqrt(3.0);
        L[7][0][0] = s3;   L[7][1][1] = s3;   L[7][2][2] = -2.0 * s3;
        for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) T[a][i][j] = 0.5 * L[a][i][j];
        for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
            cplx tr = 0.0;
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k)
                tr += (T[a][i][j] * T[b][j][k] - T[b][i][j] * T[a][j][k]) * T[c][k][i];
            cplx v = cplx(0.0, -2.0) * tr;          // -2i Tr([T^a,T^b] T^c)
            f[a][b][c] = v.real();
        }
    }
};

inline const SU3& su3() { static SU3 s; return s; }
}  // namespace orc
