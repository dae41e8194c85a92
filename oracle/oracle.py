"""ctypes front end of the CPU oracle (oracle/liboracle.so).

TEST INFRASTRUCTURE ONLY.  Allowed importers: tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  The product package
(paper_0909_5257_b200/) never imports this module and shares no code with it.

Layout of momenta: numpy float64 array of shape [n_ext, 4, n_events] (SoA), legs in
process-string order, components (E, px, py, pz) in GeV.
"""
import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_last_error.restype = C.c_char_p
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_char_p, C.c_double, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_info.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_colour_matrix.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_colour_eigenvalues.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_basis_element.restype = C.c_int
        L.orc_basis_element.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_philox.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_sample_momenta.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_uint64,
                                         C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_pass_cuts.restype = C.c_int
        L.orc_pass_cuts.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.orc_rambo_weight.restype = C.c_double
        L.orc_rambo_weight.argtypes = [C.c_int, C.c_double]
        L.orc_me2.restype = C.c_double
        L.orc_me2.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_int, C.c_int, C.c_void_p]
        L.orc_max_threads.restype = C.c_int
        L.orc_amplitudes.restype = C.c_double
        L.orc_amplitudes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_colour_sum_O1.restype = C.c_double
        L.orc_colour_sum_O1.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_bg_gluon.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.orc_gluon_colour_sum_bg.restype = C.c_double
        L.orc_gluon_colour_sum_bg.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_double]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def philox4x32_10(counter, key):
    c = np.asarray(counter, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox(_ptr(c), _ptr(k), _ptr(out))
    return out


def sample_momenta(n_final, sqrt_s, seed, n_events, first_event=0, pt_min=20.0, eta_max=2.5, dr_min=0.4):
    """Philox + massless RAMBO + cuts (steps a1-a2).  Returns (mom[n_ext,4,E], weight[E], tries[E])."""
    mom = np.zeros((n_final + 2, 4, n_events), dtype=np.float64)
    w = np.zeros(n_events, dtype=np.float64)
    tries = np.zeros(n_events, dtype=np.uint32)
    lib().orc_sample_momenta(n_final, sqrt_s, pt_min, eta_max, dr_min, seed, first_event, n_events,
                             _ptr(mom), _ptr(w), _ptr(tries))
    return mom, w, tries


def pass_cuts(p_final, pt_min=20.0, eta_max=2.5, dr_min=0.4):
    p = np.ascontiguousarray(p_final, dtype=np.float64)
    return bool(lib().orc_pass_cuts(p.shape[0], _ptr(p), pt_min, eta_max, dr_min))


def rambo_weight(n_final, sqrt_s):
    return lib().orc_rambo_weight(n_final, sqrt_s)


class Process:
    """One massless-QCD process, e.g. Process("g g > g g g", alpha_s=0.118)."""

    def __init__(self, process, alpha_s=0.118, keep_diagram_colour=False):
        self._h = lib().orc_create(process.encode(), alpha_s, int(keep_diagram_colour))
        if not self._h:
            raise RuntimeError(lib().orc_last_error().decode())
        self.process = process
        self.tier1 = bool(keep_diagram_colour)
        info = np.zeros(32)
        lib().orc_info(self._h, _ptr(info))
        self.n_ext = int(info[0])
        self.n_diagrams = int(info[1])
        self.n_topologies = int(round(info[2]))
        self.n_color = int(info[3])
        self.color_rank = int(info[4])
        self.n_pairings = int(info[5])
        self.n_nodes = int(info[6])
        self.n_assign = int(info[7])
        self.sym_factor, self.avg_color, self.avg_spin = info[8], info[9], info[10]
        self.C_max_imag, self.C_max_asym, self.max_residual = info[11], info[12], info[13]
        self.frac_nonzero_pairs, self.frac_all_zero = info[14], info[15]
        self.gs = info[16]

    def __del__(self):
        try:
            if self._h:
                lib().orc_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def colour_matrix(self):
        Cm = np.zeros((self.n_color, self.n_color))
        lib().orc_colour_matrix(self._h, _ptr(Cm))
        return Cm

    def colour_eigenvalues(self):
        ev = np.zeros(self.n_color)
        lib().orc_colour_eigenvalues(self._h, _ptr(ev))
        return ev

    def basis_element(self, alpha):
        buf = np.zeros(64, dtype=np.int32)
        lib().orc_basis_element(self._h, alpha, _ptr(buf))
        kind, pairing = int(buf[0]), int(buf[1])
        seqs, pos = [], 2
        for _ in range(4):
            n = int(buf[pos]); pos += 1
            seqs.append([int(x) for x in buf[pos:pos + n]]); pos += n
        return kind, pairing, seqs

    def me2(self, mom, tier=2, n_threads=0, return_seconds=False):
        mom = np.ascontiguousarray(mom, dtype=np.float64)
        assert mom.shape[0] == self.n_ext and mom.shape[1] == 4
        n = mom.shape[2]
        out = np.zeros(n)
        if tier == 1 and not self.tier1:
            raise RuntimeError("tier O1 needs keep_diagram_colour=True")
        sec = lib().orc_me2(self._h, _ptr(mom), n, tier, n_threads, _ptr(out))
        return (out, sec) if return_seconds else out

    def amplitudes(self, p, hel, ward_leg=-1):
        """One event p[n_ext,4], one helicity configuration -> (colour sum, J[m], A[n_diagrams])."""
        p = np.ascontiguousarray(p, dtype=np.float64)
        h = np.ascontiguousarray(hel, dtype=np.int32)
        J = np.zeros(2 * self.n_color)
        A = np.zeros(2 * self.n_diagrams)
        s = lib().orc_amplitudes(self._h, _ptr(p), _ptr(h), ward_leg, _ptr(J), _ptr(A))
        return s, J[0::2] + 1j * J[1::2], A[0::2] + 1j * A[1::2]

    def colour_sum_O1(self, p, hel):
        p = np.ascontiguousarray(p, dtype=np.float64)
        h = np.ascontiguousarray(hel, dtype=np.int32)
        return lib().orc_colour_sum_O1(self._h, _ptr(p), _ptr(h))


def bg_gluon(p, hel, order, gs):
    p = np.ascontiguousarray(p, dtype=np.float64)
    h = np.ascontiguousarray(hel, dtype=np.int32)
    o = np.ascontiguousarray(order, dtype=np.int32)
    out = np.zeros(2)
    lib().orc_bg_gluon(len(o), _ptr(p), _ptr(h), _ptr(o), gs, _ptr(out))
    return out[0] + 1j * out[1]


def gluon_colour_sum_bg(p, hel, gs):
    """sum over all 8^n colour assignments of |sum_sigma Tr(T^{c_sigma}) A_sigma|^2 for one helicity configuration of an n-gluon
    process, A_sigma from the Berends-Giele recursion (tier O1 colour on tier O3 kinematics; no diagrams, no colour basis)."""
    p = np.ascontiguousarray(p, dtype=np.float64)
    h = np.ascontiguousarray(hel, dtype=np.int32)
    return lib().orc_gluon_colour_sum_bg(p.shape[0], _ptr(p), _ptr(h), gs)


def max_threads():
    return lib().orc_max_threads()
