// heget-b200: the table program of one process (written by csrc/gen/tab.hpp, interpreted by csrc/device/heget_tab.cuh).
// Plain data, shared by the generator and the C-ABI library; see tab.hpp for what each table means.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace heget {

enum TabKindA { TA_GGG = 0, TA_GGGG = 1, TA_FUSE = 2, TA_FG = 3, TA_BG = 4 };
enum TabKindB { TB_VVV = 0, TB_GGGG = 1, TB_IOV = 2 };

struct TabProgram {
    std::string name, tag;
    int n_ext = 0, n_gluons = 0, n_quark_legs = 0;
    int n_hel_nonzero = 0, hel_weight = 1;             // configurations that do not vanish identically; 2 if the sum is parity-folded
    int NH = 0, n_hel = 0, nchunks = 0, cpc = 0;       // evaluated configurations, 2^n, warps per event, configurations per warp
    int NJ = 0, R = 0, Rpad = 0;                       // merged colour basis, rank actually accumulated, padded to tiles of 8
    int nK = 0, store32 = 0;                           // momentum slots, store size in 16-byte chunks of the FP32 layout
    int n_levels = 0, n_bundles = 0, n_bterms = 0, n_closings = 0, n_groups = 0, n_jl = 0;
    int n_diagrams = 0, n_topologies = 0, n_currents = 0, n_terms = 0, n_color = 0, n_color_eval = 0;
    double sym_factor = 1, avg_color = 1, avg_spin = 0.25;
    double flops_phase_a = 0, flops_per_hel = 0, flops_colour_per_hel = 0, flops_per_event = 0;
    // prologue
    std::vector<uint32_t> kmask;        // [nK] legs of momentum slot s (its momentum is sum of +-p over them, 1/q^2 beside it)
    std::vector<uint32_t> leginfo;      // [n]  type (0 final gluon, 1 initial gluon, 2 psi, 3 psibar) | chisign bit << 8 | stored helicities << 9 (0 both, 1 only -1, 2 only +1) | leaf base32 << 16
    // phase A (currents, once per event and variant)
    std::vector<uint32_t> a_hdr;        // [n_bundles][4]: nterms | out type << 8 | first term index << 16 ; kinds (4 bits each) ; level ; 0
    std::vector<uint32_t> a_out;        // [n_bundles][32][2]
    std::vector<uint32_t> a_term;       // [n_bterms][32][4] (word 3: index into coef)
    std::vector<uint32_t> a_level;      // [n_levels + 1] bundle ranges
    // phase B (closings, per helicity configuration)
    std::vector<uint32_t> b_rec;        // [n_entries][16] closing records (see tab.hpp)
    std::vector<uint8_t> lanerows;      // [n_rows][nchunks * 32] per-lane bytes: variant of a leg set / validity and chirality flags
    int n_entries = 0, n_rows = 0;
    std::vector<double> coef;           // pool of the distinct rational coefficients (merged-term weights, group signs, J updates)
    // phase C: colour matrix on the accumulated basis, tiles of 8 rows: cmat[(tile * Rpad + b) * 8 + i] = C[tile*8+i][b] (x2 if b > row, 0 if b < row or b >= R), plus one tile of zeros
    std::vector<double> cmat;
    // host-side info
    std::vector<int8_t> hel_table;      // [NH][n]
    std::vector<int16_t> evalidx;       // [2^n] helicity bits (leg i -> bit i, 1 = +1) -> evaluated configuration or -1
    int color_rank = 0;                 // rank of the paper-basis colour matrix
    std::vector<double> colour_paper, colour_red, colour_acc;   // paper basis; merged basis (NJ); accumulated basis (R)
};

}  // namespace heget
