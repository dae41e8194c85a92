// heget-b200: the C-ABI of include/heget.h.  Host logic only (handles, plug-in loading, argument checks, launches);
// every step of the hot path runs in the kernels of rambo.cuh (a1-a2) and of the per-process plug-ins (a3-a8).
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <set>
#include <string>
#include <vector>
#include <dlfcn.h>
#include <sys/stat.h>
#include <unistd.h>
#include "../../include/heget.h"
#include "rambo.cuh"
#include "device/heget_tab.cuh"
#include "device/heget_colour_tc.cuh"
#include "gen/tabprog.hpp"

extern "C" int heget_generate_source(const char* tag, const char* process, const char* out_path, char* msg, int msglen);
heget::TabProgram* heget_build_table(const char* tag, const char* process, int* rc, char* msg, int msglen);

namespace {

thread_local char g_err[1024] = "";
std::atomic<unsigned long long> g_launches{0};
std::mutex g_mutex;
std::map<std::string, const hg::ProcDesc*> g_plugins;      // tag -> descriptor of a loaded plug-in

heget_status_t fail(heget_status_t st, const char* fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap);
    return st;
}
#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(HEGET_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); } while (0)

std::string lib_dir() {
    Dl_info di;
    if (dladdr((void*)&heget_last_error, &di) && di.dli_fname) {
        std::string p(di.dli_fname); size_t k = p.rfind('/');
        return k == std::string::npos ? std::string(".") : p.substr(0, k);
    }
    return ".";
}
bool exists(const std::string& p) { struct stat st; return stat(p.c_str(), &st) == 0; }

// "u u~ -> g g" -> tokens {u,u~,>,g,g}; canonical name "u u~ > g g"; tag "uux_gg"
bool canonical(const char* process, std::string& name, std::string& tag, int& n_legs) {
    std::string tok; std::vector<std::string> toks;
    for (const char* c = process;; ++c) {
        if (*c == 0 || *c == ' ' || *c == '\t') { if (!tok.empty()) toks.push_back(tok); tok.clear(); if (!*c) break; }
        else tok += *c;
    }
    name.clear(); tag.clear(); n_legs = 0;
    for (size_t i = 0; i < toks.size(); ++i) {
        std::string t = toks[i]; if (t == "->") t = ">";
        if (t != ">") ++n_legs;
        if (i) name += " "; name += t;
        for (size_t k = 0; k < t.size(); ++k) {
            const char ch = t[k];
            if (ch == '>') tag += '_'; else if (ch == '~') tag += 'x';
            else if ((ch >= 'a' && ch <= 'z') || (ch >= '0' && ch <= '9')) tag += ch;
            else return false;
        }
    }
    return !toks.empty();
}

heget_status_t open_plugin(const std::string& so, const std::string& key, const std::string& name, const hg::ProcDesc** out) {
    void* h = dlopen(so.c_str(), RTLD_NOW | RTLD_LOCAL);
    if (!h) return fail(HEGET_ECOMPILE, "dlopen %s: %s", so.c_str(), dlerror());
    typedef const hg::ProcDesc* (*fn_t)();
    fn_t fn = (fn_t)dlsym(h, "heget_plugin_desc");
    if (!fn) { dlclose(h); return fail(HEGET_ECOMPILE, "%s exports no heget_plugin_desc", so.c_str()); }
    const hg::ProcDesc* d = fn();
    // a plug-in built against other headers, or one whose tag aliases another process, is refused, not misread
    if (!d || d->abi_version != HG_ABI_VERSION) { dlclose(h); return fail(HEGET_ECOMPILE, "%s was built for another version of the library: rebuild it (python -m paper_0909_5257_b200.build)", so.c_str()); }
    if (name != d->name) { dlclose(h); return fail(HEGET_EINVAL, "process '%s' is not the canonical spelling of '%s'", name.c_str(), d->name); }
    *out = g_plugins[key] = d;
    return HEGET_OK;
}

// single-quote a string for /bin/sh
std::string shq(const std::string& v) { std::string o = "'"; for (size_t i = 0; i < v.size(); ++i) { if (v[i] == '\'') o += "'\\''"; else o += v[i]; } return o + "'"; }

// One plug-in per (process, precision): kernels/heget_<tag>_f64.so / _f32.so beside this library, built ahead of time by
// paper_0909_5257_b200/build.py for the configured processes, else generated and compiled here (step a0) and cached in
// $HEGET_CACHE_DIR (default: the same kernels/ directory).
heget_status_t load_plugin(const std::string& name, const std::string& tag, int n_legs, int prec, const hg::ProcDesc** out) {
    std::lock_guard<std::mutex> lock(g_mutex);
    const std::string key = tag + (prec == 0 ? "_f64" : prec == 1 ? "_f32" : "_f32p");
    std::map<std::string, const hg::ProcDesc*>::iterator it = g_plugins.find(key);
    if (it != g_plugins.end()) { *out = it->second; return HEGET_OK; }
    const std::string dir = lib_dir() + "/kernels";
    const char* cache = getenv("HEGET_CACHE_DIR");
    const std::string wdir = cache ? std::string(cache) : dir;
    if (exists(dir + "/heget_" + key + ".so")) return open_plugin(dir + "/heget_" + key + ".so", key, name, out);
    const std::string dst = wdir + "/heget_" + key + ".so";
    if (exists(dst)) return open_plugin(dst, key, name, out);
    mkdir(wdir.c_str(), 0755);
    // intermediate files carry the pid: ranks that build the same process at the same time do not share them, and the
    // finished plug-in is moved into place atomically
    const std::string uniq = key + "." + std::to_string((long)getpid());
    const std::string cu = wdir + "/gen_" + uniq + ".cu", log = wdir + "/gen_" + uniq + ".log", tmp = dst + "." + std::to_string((long)getpid()) + ".tmp";
    char msg[512] = "";
    const int rc = heget_generate_source(tag.c_str(), name.c_str(), cu.c_str(), msg, sizeof msg);
    if (rc == 1) return fail(HEGET_EINVAL, "process '%s': %s", name.c_str(), msg);
    if (rc == 2) return fail(HEGET_EUNSUPPORTED, "process '%s': %s", name.c_str(), msg);
    if (rc != 0) return fail(HEGET_ECOMPILE, "generator failed for '%s': %s", name.c_str(), msg);
    const char* nvcc = getenv("HEGET_NVCC");
    const std::string cmd = shq(nvcc ? nvcc : "nvcc") + " -std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a -lineinfo -shared -Xcompiler -fPIC" +
                            " -DHG_ONLY_PREC=" + (prec == 0 ? "0" : prec == 1 ? "1" : "2") + (n_legs >= 6 ? " -DHG_NO_LANES1" : "") + " -I" + shq(lib_dir() + "/csrc/device") + " -o " + shq(tmp) +
                            " " + shq(cu) + " > " + shq(log) + " 2>&1";
    if (system(cmd.c_str()) != 0) return fail(HEGET_ECOMPILE, "nvcc failed for '%s' (see %s)", name.c_str(), log.c_str());
    if (rename(tmp.c_str(), dst.c_str()) != 0) return fail(HEGET_ECOMPILE, "cannot install %s", dst.c_str());
    unlink(cu.c_str());
    return open_plugin(dst, key, name, out);
}

// flat n-body massless phase-space volume (reading A7): V_n = (pi/2)^(n-1) s^(n-2) / ((n-1)! (n-2)!), times (2 pi)^(4-3n).
// Accumulated body by body: V_2 (2 pi)^-2 = 1/(8 pi), and every further particle multiplies by (pi/2) s / ((k-1)(k-2)) / (2 pi)^3.
double flat_phase_space_weight(int n, double sqrt_s) {
    const double pi = acos(-1.0), s = sqrt_s * sqrt_s;
    double w = 1.0 / (8.0 * pi);
    for (int k = 3; k <= n; ++k) w *= (pi / 2.0) * s / ((double)(k - 1) * (double)(k - 2)) / (8.0 * pi * pi * pi);
    return w;
}

// register-resident chains of dependent FMAs, 8 independent chains per thread: the measured vector-FP peak of 8(d)
template <typename T>
__global__ void __launch_bounds__(256) k_fma_probe(T* out, unsigned long long iters, T a, T b) {
    T x0 = T(threadIdx.x), x1 = x0 + T(1), x2 = x0 + T(2), x3 = x0 + T(3), x4 = x0 + T(4), x5 = x0 + T(5), x6 = x0 + T(6), x7 = x0 + T(7);
    for (unsigned long long i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

}  // namespace

struct TabShape { int epc, jm, nsp, tm_cols, tm_wcols; size_t smem; long warps; double score; };
enum TabElem { TE_F64 = 0, TE_F32 = 1, TE_F32X2 = 2 };      // element type of the table kernels: double, float, packed pair of floats (two events)
struct heget_process;
static int effective_lanes(const heget_process* p);

// One handle = one process at one precision.  Two kernel back ends can serve it (heget_set_kernel):
//   d   : the straight-line plug-in (one specialised kernel per process, generated source compiled by nvcc), loaded on demand
//   tab : the table program interpreted by the generic kernels of device/heget_tab.cuh (built in-process, no compiler)
struct heget_process {
    const hg::ProcDesc* d;
    heget::TabProgram* tab;
    int colour_stage;              // HEGET_COLOUR_* (TABLE back end)
    void* tc_x; void* tc_form; size_t tc_cap_events; const void* tc_cfull;      // tensor-core colour stage: J rows, row forms, capacity in events, full symmetric matrix
    hg::TabDev tdev; bool tab_on_device; std::vector<void*> tab_allocs; int tab_epc; TabShape tab_shape; int tab_elem;
    std::string name, tag;
    int n_legs, kernel_req;        // requested back end: HEGET_KERNEL_AUTO / STRAIGHT / TABLE
    bool auto_table;               // what AUTO means for this process
    int prec, lanes;
    double sqrt_s, alpha_s, out_scale;
    heget_cuts_t cuts;
    // scratch of the host-buffer entry point; s_mutex serialises heget_run_host calls on one handle
    double* s_mom; double* s_w; void* s_me2; size_t s_cap; std::mutex s_mutex;
};

// which back end a call takes.  AUTO: the table program for the big processes (>= 6 legs and >= 4 gluons: hundreds of
// diagrams, whose straight-line kernels are 1-3 MB of code and instruction-fetch bound), the specialised kernel otherwise
static int effective_kernel(const heget_process* p) {
    if (p->kernel_req != HEGET_KERNEL_AUTO) return p->kernel_req;
    return p->auto_table ? HEGET_KERNEL_TABLE : HEGET_KERNEL_STRAIGHT;
}

// lanes = 0 (automatic): FP64 takes the wide variant (event-cache reads become warp broadcasts; measured 26 vs 23 TFLOP/s on
// C2), FP32 the one-event-per-thread variant where it is built (the compiler keeps the event cache in registers across the
// helicity loop; measured 53 vs 40 TFLOP/s on C2)
static int effective_lanes(const heget_process* p) {
    if (p->lanes) return p->lanes;
    return (p->prec == HEGET_FP32 && (p->d->lanes_avail & 1)) ? 1 : p->d->lanes_wide;
}

// ---- the two back ends, loaded on demand -----------------------------------------------------------------------------------
static heget_status_t need_plugin(heget_process* p) {
    if (p->d) return HEGET_OK;
    return load_plugin(p->name, p->tag, p->n_legs, p->prec, &p->d);
}
static heget_status_t need_table(heget_process* p) {
    if (p->tab) return HEGET_OK;
    if (p->prec == HEGET_FP32X2) return fail(HEGET_EUNSUPPORTED, "the packed-FP32 precision exists for the straight-line kernels only");
    char msg[512] = ""; int rc = 3;
    p->tab = heget_build_table(p->tag.c_str(), p->name.c_str(), &rc, msg, sizeof msg);
    if (rc == 1) return fail(HEGET_EINVAL, "process '%s': %s", p->name.c_str(), msg);
    if (rc == 2) return fail(HEGET_EUNSUPPORTED, "process '%s': %s", p->name.c_str(), msg);
    if (rc != 0 || !p->tab) return fail(HEGET_ECOMPILE, "generator failed for '%s': %s", p->name.c_str(), msg);
    return HEGET_OK;
}
static heget_status_t need_backend(heget_process* p) { return effective_kernel(p) == HEGET_KERNEL_TABLE ? need_table(p) : need_plugin(p); }

template <typename V> static heget_status_t upload(heget_process* p, const std::vector<V>& v, const V** out) {
    void* dptr = 0;
    const size_t bytes = (v.size() ? v.size() : 1) * sizeof(V);
    if (cudaMalloc(&dptr, bytes) != cudaSuccess) { cudaGetLastError(); return fail(HEGET_ENOMEM, "cannot allocate %zu bytes of device memory for the process tables", bytes); }
    p->tab_allocs.push_back(dptr);
    if (v.size()) CU(cudaMemcpy(dptr, v.data(), v.size() * sizeof(V), cudaMemcpyHostToDevice));
    *out = (const V*)dptr;
    return HEGET_OK;
}

// Launch shape of the table kernels: events per CTA and where J lives (shared memory, or tensor memory = TMEM), chosen for the
// most resident warps per SM.  Bounds: shared memory, registers (regs per thread of the compiled kernel, 0 = unknown), 2048
// threads, and for TMEM the 512 columns of an SM (a CTA allocates a power of two >= 32; the warps of a CTA that share a
// 32-lane quadrant split the columns).  HEGET_TAB_J=smem|tmem and HEGET_TAB_EPC=n force the choice (experiments).
template <typename T> static TabShape tab_pick_shape(const hg::TabDev& d, const int (&kregs)[2][2]) {
    TabShape best; best.epc = 0; best.jm = 0; best.nsp = 1; best.tm_cols = 0; best.tm_wcols = 0; best.smem = 0; best.warps = -1; best.score = -1.0;
    const char* force = getenv("HEGET_TAB_J");
    const char* force_epc = getenv("HEGET_TAB_EPC");       // slots per CTA (experiments: the block-size scan of PAPER.md:407)
    const char* force_nsp = getenv("HEGET_TAB_NSP");       // warps per block of J (1: one warp does everything; n: n warps taking turns)
    for (int jm = 0; jm < 2; ++jm) {
        if (force && ((jm == 0) != (strcmp(force, "smem") == 0))) continue;
        for (int nsp = 1; nsp <= 4; ++nsp) for (int epc = 1; epc <= 8; ++epc) {
            const int regs = kregs[jm][nsp > 1];
            const long reg_warps = regs > 0 ? 65536 / (((regs + 7) / 8 * 8) * 32) : 64;
            if (force_epc && atoi(force_epc) != epc) continue;
            if (force_nsp && atoi(force_nsp) != nsp) continue;
            const int bwarps = epc * d.nchunks, w = bwarps * nsp, threads = w * 32;
            if (threads > (nsp == 1 ? 256 : 512) || w > reg_warps) break;
            if (nsp > 1 && (bwarps > 14 || (jm && bwarps % 4 != 0))) continue;      // named barrier per block of J; the warps that share a block of J in TMEM must sit in the same lane quadrant
            const size_t smem = hg::tab_smem_bytes<T>(d, epc, jm == 1, nsp) + 48;
            if (smem > 227 * 1024) break;
            long ctas = std::min<long>(std::min<long>((long)((228 * 1024) / (smem + 1024)), 32), 2048 / threads);
            ctas = std::min<long>(ctas, reg_warps / w);
            int cols = 0, wcols = 0;
            if (jm) {
                wcols = (int)(sizeof(T) / 4) * 2 * (d.Rpad + 1);      // + the scratch element the padded updates go to
                const int need = ((bwarps + 3) / 4) * wcols;
                cols = 32; while (cols < need) cols *= 2;
                if (cols > 512) continue;
                ctas = std::min<long>(ctas, 512 / cols);
            }
            const long warps = ctas * w;
            // what a shape is worth: blocks of J in flight, times what the warps of one block deliver together (measured: C5, g g -> 5 g,
            // u u -> u u g g g, C4; profiles/r2_block_scan.md)
            static const double gain[5] = {0.0, 1.0, 1.2, 1.6, 1.9};
            const double score = (double)(ctas * bwarps) * gain[nsp];
            // TMEM bounds the residency but the block scheduler does not know: ask for enough shared memory that no more
            // CTAs become resident than can allocate their columns (the others would spin inside tcgen05.alloc)
            size_t ask = smem;
            if (jm && ctas > 0) ask = std::max<size_t>(smem, (size_t)(228 * 1024) / (ctas + 1) + 1024 - 1024 * 1);
            if (ask > 227 * 1024) ask = 227 * 1024;
            if (score > best.score) { best.score = score; best.epc = epc; best.jm = jm; best.nsp = nsp; best.tm_cols = cols; best.tm_wcols = wcols; best.smem = ask; best.warps = warps; }
        }
    }
    return best;
}

template <typename T, int JM, bool MW> static int tab_kernel_regs() {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return 0; }
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, hg::k_tab<T, JM, MW>) != cudaSuccess) { cudaGetLastError(); return 0; }
    return fa.numRegs;
}
template <typename T> static TabShape tab_shape_T(const hg::TabDev& d) {
    const int regs[2][2] = {{tab_kernel_regs<T, 0, false>(), tab_kernel_regs<T, 0, true>()}, {tab_kernel_regs<T, 1, false>(), tab_kernel_regs<T, 1, true>()}};      // [J in TMEM][several warps per J]
    return tab_pick_shape<T>(d, regs);
}
// FP32 handles run the table program on packed f32x2 arithmetic, two events per warp (HEGET_TAB_PACK=0: scalar, one event per warp)
static int tab_elem_of(int prec) {
    if (prec == HEGET_FP64) return TE_F64;
    const char* e = getenv("HEGET_TAB_PACK");
    return (e && e[0] == '0') ? TE_F32 : TE_F32X2;
}
static TabShape tab_shape_of(const hg::TabDev& d, int elem) {
    if (elem == TE_F64) return tab_shape_T<double>(d);
    if (elem == TE_F32) return tab_shape_T<float>(d);
    return tab_shape_T<hg::f2>(d);
}

static heget_status_t table_to_device(heget_process* p) {
    if (p->tab_on_device) return HEGET_OK;
    p->tab_elem = tab_elem_of(p->prec);
    const heget::TabProgram& t = *p->tab;
    hg::TabDev& d = p->tdev;
    memset(&d, 0, sizeof d);
    d.n_ext = t.n_ext; d.NH = t.NH; d.nchunks = t.nchunks; d.cpc = t.cpc; d.R = t.R; d.Rpad = t.Rpad; d.nK = t.nK; d.store32 = t.store32;
    d.n_levels = t.n_levels; d.n_closings = t.n_closings;
    heget_status_t st;
    if ((st = upload(p, t.kmask, &d.kmask)) != HEGET_OK) return st;
    if ((st = upload(p, t.leginfo, &d.leginfo)) != HEGET_OK) return st;
    if ((st = upload(p, t.a_hdr, &d.a_hdr)) != HEGET_OK) return st;
    if ((st = upload(p, t.a_out, &d.a_out)) != HEGET_OK) return st;
    if ((st = upload(p, t.a_term, &d.a_term)) != HEGET_OK) return st;
    if ((st = upload(p, t.a_level, &d.a_level)) != HEGET_OK) return st;
    {   // closing records in the byte layout of this precision (heget_tab.cuh, tab_load_ops / tab_finish)
        const bool f64 = p->tab_elem != TE_F32;       // 8-byte elements: double, or a pair of floats
        const bool pairf = p->tab_elem == TE_F32X2;
        auto enc8 = [&](double c, void* dst) { if (pairf) { const float f[2] = {(float)c, (float)c}; memcpy(dst, f, 8); } else memcpy(dst, &c, 8); };
        const unsigned scale = f64 ? 2u : 1u, esz = f64 ? 8u : 4u;
        const size_t ENT = f64 ? hg::tab_entry_bytes<double>() : hg::tab_entry_bytes<float>(), LT = (size_t)t.nchunks * 32;
        // launch shape first: with nsp > 1 warps per block of J (heget_tab.cuh) every warp walks its own list of records, the colour groups
        // dealt out gpt at a time in turn; every list is padded with null records for the read-ahead of its ring
        d.n_rows = t.n_rows; d.n_entries = t.n_entries;
        p->tab_shape = tab_shape_of(d, p->tab_elem);
        if (p->tab_shape.epc == 0) return fail(HEGET_EUNSUPPORTED, "process '%s': one event does not fit the shared memory of an SM", p->name.c_str());
        d.nsp = p->tab_shape.nsp; d.gpt = 2;
        { const char* e = getenv("HEGET_TAB_GPT"); if (e && atoi(e) >= 1 && atoi(e) <= 64) d.gpt = atoi(e); }      // colour groups a producer takes per turn (experiments)
        const int nlists = d.nsp > 1 ? d.nsp : 1;
        std::vector<int> seq;
        {
            std::vector<std::vector<int> > lists(nlists);
            int g = 0;
            for (int k = 0; k < t.n_entries; ++k) {
                lists[(g / d.gpt) % nlists].push_back(k);
                const uint32_t e0 = t.b_rec[(size_t)k * 16];
                if ((e0 >> 2) & 1u) { ++g; if (((e0 >> 3) & 15u) == 0u) return fail(HEGET_EUNSUPPORTED, "process '%s': a colour group without updates", p->name.c_str()); }      // the turn passing counts groups by their last update record
            }
            for (int l = 0; l < nlists; ++l) {
                d.list0[l] = (int)seq.size(); d.nrec[l] = (int)lists[l].size(); d.ngrp[l] = 0;
                for (size_t i = 0; i < lists[l].size(); ++i) { seq.push_back(lists[l][i]); if ((t.b_rec[(size_t)lists[l][i] * 16] >> 2) & 1u) ++d.ngrp[l]; }
                for (int i = 0; i < HG_TAB_RING + 2; ++i) seq.push_back(-1);
            }
        }
        const size_t npad = seq.size();
        std::vector<unsigned char> ent(npad * ENT, 0);
        for (size_t k = 0; k < npad; ++k) {
            uint32_t w[48]; memset(w, 0, sizeof w);
            if (seq[k] < 0) { w[0] = 3u; memcpy(&ent[k * ENT], w, ENT); continue; }      // null record: no amplitude, no update
            const uint32_t* e = &t.b_rec[(size_t)seq[k] * 16];
            const unsigned kind = e[0] & 3u, reset = (e[0] >> 2) & 1u, nu = (e[0] >> 3) & 15u;
            const unsigned base[4] = {e[1] & 0xffffu, e[1] >> 16, e[2] & 0xffffu, e[2] >> 16};
            unsigned row[4], stride[4];
            for (int j = 0; j < 4; ++j) { row[j] = ((e[3] >> (8 * j)) & 0xffu) * (unsigned)LT; stride[j] = 1u << ((e[0] >> (8 + 3 * j)) & 7u); if (scale * base[j] > 0xffffu || row[j] > 0xffffu) return fail(HEGET_EUNSUPPORTED, "process '%s': current store too large for the table format", p->name.c_str()); }
            const unsigned frow = (e[4] & 0xffu) * (unsigned)LT, ka = ((e[4] >> 8) & 0xffu) * 4u * esz, kb = ((e[4] >> 16) & 0xffu) * 4u * esz;
            if (frow > 0xffffu || ka > 0xffffu || kb > 0xffffu) return fail(HEGET_EUNSUPPORTED, "process '%s': tables too large for the record format", p->name.c_str());
            w[0] = kind | (reset << 2) | (nu << 3) | (frow << 16);
            w[1] = scale * base[0] | (scale * base[1] << 16); w[2] = scale * base[2] | (scale * base[3] << 16);
            w[3] = row[0] | (row[1] << 16); w[4] = row[2] | (row[3] << 16);
            w[5] = stride[0] | (stride[1] << 8) | (stride[2] << 16) | (stride[3] << 24);
            w[6] = ka | (kb << 16);
            const double sgn = t.coef[e[5]];
            if (f64) {
                enc8(sgn, &w[8]);
                for (unsigned j = 0; j < nu; ++j) { const double c = t.coef[e[6 + j] >> 16]; w[12 + 4 * j] = (e[6 + j] & 0xffffu) * 2u * 32u * 8u; enc8(c, &w[14 + 4 * j]); }
                for (unsigned j = nu; j < (nu + 3u) / 4u * 4u; ++j) { w[12 + 4 * j] = (unsigned)t.Rpad * 2u * 32u * 8u; enc8(0.0, &w[14 + 4 * j]); }      // pads: scratch element, coefficient 0 (branch-free batches, JTmem::update)
            } else {
                const float sf = (float)sgn; memcpy(&w[7], &sf, 4);
                for (unsigned j = 0; j < nu; ++j) { const float c = (float)t.coef[e[6 + j] >> 16]; w[8 + 2 * j] = (e[6 + j] & 0xffffu) * 2u * 32u * 4u; memcpy(&w[9 + 2 * j], &c, 4); }      // 8 x {offset, coefficient} from byte 32
                for (unsigned j = nu; j < (nu + 3u) / 4u * 4u; ++j) { w[8 + 2 * j] = (unsigned)t.Rpad * 2u * 32u * 4u; w[9 + 2 * j] = 0u; }
            }
            memcpy(&ent[k * ENT], w, ENT);
        }
        if ((st = upload(p, ent, &d.b_ent)) != HEGET_OK) return st;
        std::vector<unsigned char> rows(t.lanerows.begin(), t.lanerows.end()); rows.resize((rows.size() + 15) / 16 * 16 + 16, 0);
        if ((st = upload(p, rows, &d.lanerows)) != HEGET_OK) return st;
        d.n_entries = t.n_entries; d.n_rows = t.n_rows;
    }
    if ((st = upload(p, t.evalidx, &d.evalidx)) != HEGET_OK) return st;
    // colour stage: what the tiles hold (heget_tab.cuh, phase C)
    std::vector<double> cmat = t.cmat;
    d.cstage = 0; d.cidx = 0; d.cvals = 0;
    std::vector<double> cvals; std::vector<unsigned char> cidx;
    if (p->colour_stage == HEGET_COLOUR_CHOLESKY) {
        // C = L L^T (C is positive semi-definite; a vanishing pivot means the rest of its column vanishes too): rows of L^T in the tile layout
        const int R = t.R, Rp = t.Rpad;
        std::vector<double> L((size_t)R * R, 0.0);
        for (int j = 0; j < R; ++j) {
            double dj = t.colour_acc[(size_t)j * R + j];
            for (int k = 0; k < j; ++k) dj -= L[(size_t)j * R + k] * L[(size_t)j * R + k];
            if (dj <= 1e-12 * t.colour_acc[(size_t)j * R + j]) continue;       // null direction: column j of L stays zero
            const double lj = sqrt(dj); L[(size_t)j * R + j] = lj;
            for (int i = j + 1; i < R; ++i) {
                double v = t.colour_acc[(size_t)i * R + j];
                for (int k = 0; k < j; ++k) v -= L[(size_t)i * R + k] * L[(size_t)j * R + k];
                L[(size_t)i * R + j] = v / lj;
            }
        }
        std::fill(cmat.begin(), cmat.end(), 0.0);
        for (int tl = 0; tl < Rp / 8; ++tl) for (int b = 0; b < R; ++b) for (int i = 0; i < 8; ++i) { const int a = tl * 8 + i; if (a < R && b >= a) cmat[((size_t)tl * Rp + b) * 8 + i] = L[(size_t)b * R + a]; }
        d.cstage = 2;
    } else if (p->colour_stage == HEGET_COLOUR_TENSOR) {
        if (t.Rpad > 8 * hg::TC_MAX_NT) return fail(HEGET_EUNSUPPORTED, "process '%s': the tensor-core colour stage takes at most %d colour elements", p->name.c_str(), 8 * hg::TC_MAX_NT);
        // the full symmetric matrix, padded with zeros to Rpad x Rpad, in the precision of the contraction
        const int R = t.R, Rp = t.Rpad;
        if (p->prec == HEGET_FP64) { std::vector<double> cfull((size_t)Rp * Rp, 0.0); for (int a = 0; a < R; ++a) for (int b = 0; b < R; ++b) cfull[(size_t)a * Rp + b] = t.colour_acc[(size_t)a * R + b]; const double* c = 0; if ((st = upload(p, cfull, &c)) != HEGET_OK) return st; p->tc_cfull = c; }
        else { std::vector<float> cfull((size_t)Rp * Rp, 0.f); for (int a = 0; a < R; ++a) for (int b = 0; b < R; ++b) cfull[(size_t)a * Rp + b] = (float)t.colour_acc[(size_t)a * R + b]; const float* c = 0; if ((st = upload(p, cfull, &c)) != HEGET_OK) return st; p->tc_cfull = c; }
        d.cstage = 3;
    } else if (p->colour_stage == HEGET_COLOUR_DISTINCT) {
        std::map<double, int> index;
        cidx.assign(cmat.size() + 64, 0);
        for (size_t i = 0; i < cmat.size(); ++i) {
            std::map<double, int>::iterator it = index.find(cmat[i]);
            if (it == index.end()) { const int id = (int)cvals.size(); if (id > 255) return fail(HEGET_EUNSUPPORTED, "process '%s': more than 256 distinct colour coefficients", p->name.c_str()); index[cmat[i]] = id; cvals.push_back(cmat[i]); cidx[i] = (unsigned char)id; }
            else cidx[i] = (unsigned char)it->second;
        }
        if ((st = upload(p, cidx, &d.cidx)) != HEGET_OK) return st;
        d.cstage = 1;
    }
    if (p->tab_elem == TE_F64) {
        const double* c = 0; if ((st = upload(p, cmat, &c)) != HEGET_OK) return st; d.cmat = c;
        if ((st = upload(p, t.coef, &c)) != HEGET_OK) return st; d.coef = c;
        if (d.cstage == 1) { if ((st = upload(p, cvals, &c)) != HEGET_OK) return st; d.cvals = c; }
    } else if (p->tab_elem == TE_F32) {
        std::vector<float> cm(cmat.begin(), cmat.end()), cf(t.coef.begin(), t.coef.end()), cv(cvals.begin(), cvals.end()); const float* c = 0;
        if ((st = upload(p, cm, &c)) != HEGET_OK) return st; d.cmat = c;
        if ((st = upload(p, cf, &c)) != HEGET_OK) return st; d.coef = c;
        if (d.cstage == 1) { if ((st = upload(p, cv, &c)) != HEGET_OK) return st; d.cvals = c; }
    } else {      // both halves of a packed value hold the same coefficient
        std::vector<float> cm(2 * cmat.size()), cf(2 * t.coef.size()), cv(2 * cvals.size()); const float* c = 0;
        for (size_t i = 0; i < cmat.size(); ++i) cm[2 * i] = cm[2 * i + 1] = (float)cmat[i];
        for (size_t i = 0; i < t.coef.size(); ++i) cf[2 * i] = cf[2 * i + 1] = (float)t.coef[i];
        for (size_t i = 0; i < cvals.size(); ++i) cv[2 * i] = cv[2 * i + 1] = (float)cvals[i];
        if ((st = upload(p, cm, &c)) != HEGET_OK) return st; d.cmat = c;
        if ((st = upload(p, cf, &c)) != HEGET_OK) return st; d.coef = c;
        if (d.cstage == 1) { if ((st = upload(p, cv, &c)) != HEGET_OK) return st; d.cvals = c; }
    }
    p->tab_epc = p->tab_shape.epc;
    const int smem = (int)p->tab_shape.smem;
#define HG_TAB_ATTR2(TT, JMV) do { if (p->tab_shape.nsp > 1) CU(cudaFuncSetAttribute(hg::k_tab<TT, JMV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); else CU(cudaFuncSetAttribute(hg::k_tab<TT, JMV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); } while (0)
#define HG_TAB_ATTR(TT) do { if (p->tab_shape.jm) HG_TAB_ATTR2(TT, 1); else HG_TAB_ATTR2(TT, 0); } while (0)
    if (p->tab_elem == TE_F64) HG_TAB_ATTR(double);
    else if (p->tab_elem == TE_F32) HG_TAB_ATTR(float);
    else HG_TAB_ATTR(hg::f2);
#undef HG_TAB_ATTR
#undef HG_TAB_ATTR2
    p->tab_on_device = true;
    return HEGET_OK;
}

static void table_free_device(heget_process* p) {
    for (size_t i = 0; i < p->tab_allocs.size(); ++i) cudaFree(p->tab_allocs[i]);
    p->tab_allocs.clear(); p->tab_on_device = false;
}

extern "C" {

const char* heget_last_error(void) { return g_err; }
uint64_t heget_launch_count(void) { return g_launches.load(); }
#ifdef HG_TAB_TIMING
void heget_debug_timing(unsigned long long* out, int reset) { cudaDeviceSynchronize(); cudaMemcpyFromSymbol(out, hg::g_tab_timing, 128); if (reset) { unsigned long long z[16] = {0}; cudaMemcpyToSymbol(hg::g_tab_timing, z, 128); } }
#endif

heget_status_t heget_fma_probe(heget_precision_t prec, uint64_t iters, void* d_out, uint64_t n_threads, double* flops, void* cuda_stream) {
    if (!d_out || !flops || n_threads == 0 || n_threads % 256) return fail(HEGET_EINVAL, "heget_fma_probe: d_out/flops NULL or n_threads not a multiple of 256");
    const unsigned int blocks = (unsigned int)(n_threads / 256);
    if (prec == HEGET_FP64) k_fma_probe<double><<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>((double*)d_out, iters, 0.999999, 1e-6);
    else if (prec == HEGET_FP32) k_fma_probe<float><<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>((float*)d_out, iters, 0.9999f, 1e-4f);
    else return fail(HEGET_EINVAL, "heget_fma_probe: unknown precision");
    CU(cudaGetLastError());
    *flops = 16.0 * (double)iters * (double)n_threads;
    return HEGET_OK;
}

heget_status_t heget_process_create(const char* process, double sqrt_s_hat, double alpha_s, const heget_cuts_t* cuts,
                                    heget_precision_t prec, heget_process_t** out) {
    if (!process || !out) return fail(HEGET_EINVAL, "heget_process_create: NULL argument");
    if (!(sqrt_s_hat > 0.0) || !(alpha_s > 0.0) || !std::isfinite(sqrt_s_hat) || !std::isfinite(alpha_s))
        return fail(HEGET_EINVAL, "heget_process_create: sqrt_s_hat and alpha_s must be positive and finite");
    if (prec != HEGET_FP64 && prec != HEGET_FP32 && prec != HEGET_FP32X2) return fail(HEGET_EINVAL, "heget_process_create: unknown precision %d", (int)prec);
    std::string name, tag; int n_legs = 0;
    if (!canonical(process, name, tag, n_legs)) return fail(HEGET_EINVAL, "heget_process_create: cannot parse process '%s'", process);
    if (prec == HEGET_FP32X2 && (" " + name + " ").find(" g ") == std::string::npos)
        return fail(HEGET_EUNSUPPORTED, "process '%s' has no gluon whose two helicities could share a packed thread", name.c_str());
    heget_process* p = new (std::nothrow) heget_process();
    if (!p) return fail(HEGET_ENOMEM, "out of host memory");
    p->d = 0; p->tab = 0; p->tab_on_device = false; p->tab_epc = 0; p->colour_stage = HEGET_COLOUR_SYMMETRIC; p->tc_x = 0; p->tc_form = 0; p->tc_cap_events = 0; p->tc_cfull = 0; p->name = name; p->tag = tag; p->n_legs = n_legs;
    p->kernel_req = prec == HEGET_FP32X2 ? HEGET_KERNEL_STRAIGHT : HEGET_KERNEL_AUTO;
    { int ng = 0; const std::string padded = " " + name + " "; for (size_t q = 0; q + 2 < padded.size(); ++q) if (padded[q] == ' ' && padded[q + 1] == 'g' && padded[q + 2] == ' ') ++ng; p->auto_table = n_legs >= 7 || (n_legs == 6 && ng >= 6); }
    p->prec = (int)prec; p->lanes = 0; p->sqrt_s = sqrt_s_hat; p->alpha_s = alpha_s;
    p->cuts.pt_min = cuts ? cuts->pt_min : 0.0; p->cuts.eta_max = cuts ? cuts->eta_max : 0.0; p->cuts.dr_min = cuts ? cuts->dr_min : 0.0;
    p->s_mom = 0; p->s_w = 0; p->s_me2 = 0; p->s_cap = 0;
    const heget_status_t st = need_backend(p);
    if (st != HEGET_OK) { delete p; return st; }
    // S * 1/4 * 1/(n_a n_b) * g_s^(2(n-2)) * s_hat^-(n-4): the kernels work in units of sqrt(s_hat) (reading A21)
    const double gs2 = 4.0 * 3.14159265358979323846 * alpha_s;
    const double sym = p->tab ? p->tab->sym_factor : p->d->sym_factor, avs = p->tab ? p->tab->avg_spin : p->d->avg_spin, avc = p->tab ? p->tab->avg_color : p->d->avg_color;
    p->out_scale = sym * avs * avc * pow(gs2, n_legs - 2) * pow(sqrt_s_hat, -2.0 * (n_legs - 4));
    *out = p;
    return HEGET_OK;
}

void heget_destroy(heget_process_t* p) {
    if (!p) return;
    if (p->s_mom) cudaFree(p->s_mom);
    if (p->s_w) cudaFree(p->s_w);
    if (p->s_me2) cudaFree(p->s_me2);
    if (p->tc_x) cudaFree(p->tc_x);
    if (p->tc_form) cudaFree(p->tc_form);
    table_free_device(p);
    delete p->tab;
    delete p;
}

heget_status_t heget_set_kernel(heget_process_t* p, heget_kernel_t kernel) {
    if (!p) return fail(HEGET_EINVAL, "heget_set_kernel: NULL handle");
    if (kernel != HEGET_KERNEL_AUTO && kernel != HEGET_KERNEL_STRAIGHT && kernel != HEGET_KERNEL_TABLE) return fail(HEGET_EINVAL, "heget_set_kernel: unknown back end %d", (int)kernel);
    if (p->prec == HEGET_FP32X2 && kernel == HEGET_KERNEL_TABLE) return fail(HEGET_EUNSUPPORTED, "the packed-FP32 precision exists for the straight-line kernels only");
    const int old = p->kernel_req;
    p->kernel_req = p->prec == HEGET_FP32X2 ? HEGET_KERNEL_STRAIGHT : (int)kernel;
    const heget_status_t st = need_backend(p);
    if (st != HEGET_OK) p->kernel_req = old;
    return st;
}

heget_status_t heget_set_colour_stage(heget_process_t* p, heget_colour_stage_t stage) {
    if (!p) return fail(HEGET_EINVAL, "heget_set_colour_stage: NULL handle");
    if (stage != HEGET_COLOUR_SYMMETRIC && stage != HEGET_COLOUR_DISTINCT && stage != HEGET_COLOUR_CHOLESKY && stage != HEGET_COLOUR_TENSOR) return fail(HEGET_EINVAL, "heget_set_colour_stage: unknown stage %d", (int)stage);
    if (effective_kernel(p) != HEGET_KERNEL_TABLE) return fail(HEGET_EUNSUPPORTED, "heget_set_colour_stage: the straight-line kernels carry their colour form as literal code; select the TABLE back end first");
    if ((int)stage != p->colour_stage) { p->colour_stage = (int)stage; table_free_device(p); }      // the tiles are rebuilt at the next launch
    return HEGET_OK;
}

heget_status_t heget_set_lanes(heget_process_t* p, int lanes) {
    if (!p) return fail(HEGET_EINVAL, "heget_set_lanes: NULL handle");
    if (effective_kernel(p) == HEGET_KERNEL_TABLE) {
        if (lanes != 0 && lanes != 32) return fail(HEGET_EINVAL, "heget_set_lanes: the table kernels have one layout (a warp per 32 helicity configurations); lanes must be 0 or 32");
        p->lanes = 0; return HEGET_OK;
    }
    const hg::ProcDesc* d = p->d;
    const bool ok = lanes == 0 || (lanes == 1 && (d->lanes_avail & 1)) || (lanes == d->lanes_wide && (d->lanes_avail & 2));
    if (!ok) return fail(HEGET_EINVAL, "heget_set_lanes: lanes = %d is not built for '%s' (0 = automatic%s, wide = %d)", lanes, d->name,
                         (d->lanes_avail & 1) ? ", 1" : "", d->lanes_wide);
    p->lanes = lanes; return HEGET_OK;
}

heget_status_t heget_process_info(const heget_process_t* p, heget_info_t* o) {
    if (!p || !o) return fail(HEGET_EINVAL, "heget_process_info: NULL argument");
    memset(o, 0, sizeof *o);
    o->regs_per_thread = -1; o->local_bytes_per_thread = -1; o->color_rank = -1;
    int ndev = 0;
    const bool have_dev = cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0;
    if (!have_dev) cudaGetLastError();
    if (effective_kernel(p) == HEGET_KERNEL_TABLE) {
        const heget::TabProgram& t = *p->tab;
        o->kernel = HEGET_KERNEL_TABLE;
        o->n_ext = t.n_ext; o->n_hel = t.n_hel; o->n_hel_eval = t.n_hel_nonzero; o->n_hel_computed = t.NH; o->n_diagrams = t.n_diagrams; o->n_topologies = t.n_topologies;
        o->n_color = t.n_color; o->n_color_eval = t.n_color_eval; o->n_color_reduced = t.NJ; o->n_color_accum = t.R; o->color_rank = t.color_rank;
        o->avg_spin = t.avg_spin; o->avg_color = t.avg_color; o->sym_factor = t.sym_factor;
        o->flops_per_event = t.flops_per_event; o->flops_per_helicity = t.flops_per_hel;
        o->lanes_wide = 32; o->lanes = 32;
        hg::TabDev d; memset(&d, 0, sizeof d); d.n_ext = t.n_ext; d.nchunks = t.nchunks; d.R = t.R; d.nK = t.nK; d.store32 = t.store32; d.n_rows = t.n_rows;
        d.Rpad = t.Rpad;
        const int elem = tab_elem_of(p->prec);
        const TabShape sh = tab_shape_of(d, elem);
        o->events_per_block = sh.epc * (elem == TE_F32X2 ? 2 : 1); o->threads_per_block = sh.epc * t.nchunks * 32 * sh.nsp; o->j_in_tmem = sh.jm; o->warps_per_j = sh.nsp; o->packed_pairs = elem == TE_F32X2; o->colour_stage = p->colour_stage;
        { std::set<long long> dv; for (size_t i = 0; i < t.colour_acc.size(); ++i) if (t.colour_acc[i] != 0.0) dv.insert((long long)llround(t.colour_acc[i] * 1e9)); o->n_color_distinct = (int)dv.size(); }
        if (have_dev) {
            cudaFuncAttributes fa;
            cudaError_t e;
#define HG_TAB_FA(TT) (sh.jm ? (sh.nsp > 1 ? cudaFuncGetAttributes(&fa, hg::k_tab<TT, 1, true>) : cudaFuncGetAttributes(&fa, hg::k_tab<TT, 1, false>)) : (sh.nsp > 1 ? cudaFuncGetAttributes(&fa, hg::k_tab<TT, 0, true>) : cudaFuncGetAttributes(&fa, hg::k_tab<TT, 0, false>)))
            if (elem == TE_F64) e = HG_TAB_FA(double); else if (elem == TE_F32) e = HG_TAB_FA(float); else e = HG_TAB_FA(hg::f2);
#undef HG_TAB_FA
            if (e == cudaSuccess) { o->regs_per_thread = fa.numRegs; o->local_bytes_per_thread = (int)fa.localSizeBytes; } else cudaGetLastError();
        }
        return HEGET_OK;
    }
    const hg::ProcDesc* d = p->d;
    o->kernel = HEGET_KERNEL_STRAIGHT;
    o->n_ext = d->n_ext; o->n_hel = d->n_hel; o->n_hel_eval = d->n_hel_eval; o->n_hel_computed = d->n_hel_eval; o->n_diagrams = d->n_diagrams; o->n_topologies = d->n_topologies;
    o->n_color = d->n_color; o->n_color_eval = d->n_color_eval; o->n_color_reduced = d->n_color_reduced; o->n_color_accum = d->n_color_reduced;
    if (p->tab) o->color_rank = p->tab->color_rank;
    o->avg_spin = d->avg_spin; o->avg_color = d->avg_color; o->sym_factor = d->sym_factor;
    o->flops_per_event = d->flops_per_event; o->flops_per_helicity = d->flops_per_hel;
    o->threads_per_block = d->block[p->prec == HEGET_FP64 ? 0 : 1]; o->lanes_wide = d->lanes_wide; o->lanes = effective_lanes(p);
    o->events_per_block = o->threads_per_block / o->lanes;
    if (have_dev) {
        hg::KernelInfo ki;
        if (d->kernel_info(p->prec, effective_lanes(p), &ki) == 0) { o->regs_per_thread = ki.regs; o->local_bytes_per_thread = ki.local_bytes; o->threads_per_block = ki.block; o->events_per_block = ki.block / o->lanes; }
        else cudaGetLastError();
    }
    return HEGET_OK;
}

heget_status_t heget_color_matrix(const heget_process_t* p, int which, double* h_out, int* n) {
    if (!p || !n) return fail(HEGET_EINVAL, "heget_color_matrix: NULL argument");
    if (which < 0 || which > 2) return fail(HEGET_EINVAL, "heget_color_matrix: which must be 0, 1 or 2");
    if (effective_kernel(p) == HEGET_KERNEL_TABLE) {
        const heget::TabProgram& t = *p->tab;
        const std::vector<double>& c = which == 0 ? t.colour_paper : which == 1 ? t.colour_red : t.colour_acc;
        const int m = which == 0 ? t.n_color : which == 1 ? t.NJ : t.R;
        *n = m;
        if (h_out) memcpy(h_out, c.data(), sizeof(double) * (size_t)m * m);
        return HEGET_OK;
    }
    const int m = which == 0 ? p->d->n_color : p->d->n_color_reduced;
    *n = m;
    if (h_out) memcpy(h_out, which == 0 ? p->d->colour_matrix : p->d->colour_matrix_eval, sizeof(double) * (size_t)m * m);
    return HEGET_OK;
}

heget_status_t heget_sample_momenta(heget_process_t* p, uint64_t seed, uint64_t first_event, uint64_t n_events,
                                    double* d_mom, double* d_weight, uint32_t* d_tries, void* cuda_stream) {
    if (!p) return fail(HEGET_EINVAL, "heget_sample_momenta: NULL handle");
    if (n_events == 0) return HEGET_OK;
    if (!d_mom) return fail(HEGET_EINVAL, "heget_sample_momenta: d_mom is NULL");
    if (n_events > (1ull << 31) * 128ull) return fail(HEGET_EINVAL, "heget_sample_momenta: n_events too large");
    const int nf = p->n_legs - 2;
    hg::RamboArgs a;
    a.sqrt_s = p->sqrt_s; a.pt_min = p->cuts.pt_min; a.eta_max = p->cuts.eta_max; a.dr_min = p->cuts.dr_min;
    a.w0 = flat_phase_space_weight(nf, p->sqrt_s);
    a.seed = seed; a.first_event = first_event; a.n_events = n_events; a.mom = d_mom; a.weight = d_weight; a.tries = d_tries;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const unsigned int blocks = (unsigned int)((n_events + 127) / 128);
    switch (nf) {
        case 2: hg::k_rambo<2><<<blocks, 128, 0, s>>>(a); break;
        case 3: hg::k_rambo<3><<<blocks, 128, 0, s>>>(a); break;
        case 4: hg::k_rambo<4><<<blocks, 128, 0, s>>>(a); break;
        case 5: hg::k_rambo<5><<<blocks, 128, 0, s>>>(a); break;
        case 6: hg::k_rambo<6><<<blocks, 128, 0, s>>>(a); break;
        default: return fail(HEGET_EUNSUPPORTED, "heget_sample_momenta: %d final-state particles", nf);
    }
    CU(cudaGetLastError());
    g_launches++;
    return HEGET_OK;
}

heget_status_t heget_eval_me2(heget_process_t* p, const double* d_mom, uint64_t n_events, heget_hel_mode_t mode,
                              const int8_t* hel, uint64_t seed, uint64_t first_event, void* d_me2, void* cuda_stream) {
    if (!p) return fail(HEGET_EINVAL, "heget_eval_me2: NULL handle");
    if (mode != HEGET_HEL_SUM && mode != HEGET_HEL_SAMPLE && mode != HEGET_HEL_FIXED) return fail(HEGET_EINVAL, "heget_eval_me2: unknown helicity mode %d", (int)mode);
    if (mode == HEGET_HEL_FIXED && !hel) return fail(HEGET_EINVAL, "heget_eval_me2: HEL_FIXED needs hel");
    if (n_events == 0) return HEGET_OK;
    if (!d_mom || !d_me2) return fail(HEGET_EINVAL, "heget_eval_me2: NULL device pointer");
    const bool table = effective_kernel(p) == HEGET_KERNEL_TABLE;
    const int n_ext = p->n_legs;
    const int n_eval = table ? p->tab->NH : p->d->n_hel_eval;
    const signed char* htab = table ? (const signed char*)p->tab->hel_table.data() : p->d->hel_table;
    int hel_fixed = -1;
    if (mode == HEGET_HEL_FIXED) {
        for (int i = 0; i < n_ext; ++i) if (hel[i] != 1 && hel[i] != -1) return fail(HEGET_EINVAL, "heget_eval_me2: hel[%d] = %d is not +-1", i, (int)hel[i]);
        const bool folded = table && p->tab->hel_weight == 2;
        for (int h = 0; h < n_eval && hel_fixed < 0; ++h) {
            bool same = true, mirror = folded;
            for (int i = 0; i < n_ext; ++i) { if (htab[h * n_ext + i] != hel[i]) same = false; if (htab[h * n_ext + i] != -hel[i]) mirror = false; }
            if (same || mirror) hel_fixed = h;
        }
    }
    if (table) {
        const heget_status_t st = table_to_device(p);
        if (st != HEGET_OK) return st;
        const int epc = p->tab_epc;
        const int evpc = epc * (p->tab_elem == TE_F32X2 ? 2 : 1);       // events per CTA
        const unsigned long long blocks = (n_events + evpc - 1) / evpc;
        if (blocks > 0x7fffffffull) return fail(HEGET_EINVAL, "heget_eval_me2: n_events too large for one launch");
        const int threads = epc * p->tdev.nchunks * 32 * p->tdev.nsp;
        cudaStream_t s = (cudaStream_t)cuda_stream;
        const TabShape& sh = p->tab_shape;
        const double iss = 1.0 / p->sqrt_s;
        // parity-folded helicity sum: every evaluated configuration stands for itself and its mirror image
        const double oscale = p->out_scale * (mode == HEGET_HEL_SUM ? (double)p->tab->hel_weight : 1.0);
#define HG_TAB_LAUNCH3(TT, OT, JMV, MWV) hg::k_tab<TT, JMV, MWV><<<(unsigned int)cblocks, threads, sh.smem, s>>>(dev, epc, sh.tm_cols, sh.tm_wcols, d_mom + first, n_events, count, iss, oscale, (OT*)d_me2 + first, (int)mode, hel_fixed, seed, first_event + first)
        hg::TabDev dev = p->tdev;
        const bool tensor = dev.cstage == 3;
        unsigned long long chunk = n_events;
        const size_t esz = p->prec == HEGET_FP64 ? 8 : 4;
        const size_t rows_per_event = (size_t)dev.nchunks * 32 * 2;
        if (tensor) {
            if (mode != HEGET_HEL_SUM) return fail(HEGET_EUNSUPPORTED, "heget_eval_me2: the tensor-core colour stage serves HEL_SUM only");
            // J rows go through HBM in chunks of at most 1 GiB
            const size_t per_event = rows_per_event * dev.Rpad * esz;
            chunk = std::max<unsigned long long>(evpc, std::min<unsigned long long>(n_events, ((size_t)1 << 30) / per_event / evpc * evpc));
            if (p->tc_cap_events < chunk) {
                if (p->tc_x) cudaFree(p->tc_x); if (p->tc_form) cudaFree(p->tc_form);
                p->tc_x = 0; p->tc_form = 0; p->tc_cap_events = 0;
                if (cudaMalloc(&p->tc_x, chunk * per_event) != cudaSuccess || cudaMalloc(&p->tc_form, chunk * rows_per_event * esz) != cudaSuccess) { cudaGetLastError(); return fail(HEGET_ENOMEM, "heget_eval_me2: cannot allocate the J buffer of the tensor-core colour stage"); }
                p->tc_cap_events = chunk;
            }
            dev.jout = p->tc_x;
        }
        for (unsigned long long first = 0; first < n_events; first += chunk) {
            const unsigned long long count = std::min<unsigned long long>(chunk, n_events - first);
            const unsigned long long cblocks = (count + evpc - 1) / evpc;
#define HG_TAB_LAUNCH2(TT, OT, JMV) do { if (sh.nsp > 1) HG_TAB_LAUNCH3(TT, OT, JMV, true); else HG_TAB_LAUNCH3(TT, OT, JMV, false); } while (0)
#define HG_TAB_LAUNCH(TT, OT) do { if (sh.jm) HG_TAB_LAUNCH2(TT, OT, 1); else HG_TAB_LAUNCH2(TT, OT, 0); } while (0)
            if (p->tab_elem == TE_F64) HG_TAB_LAUNCH(double, double);
            else if (p->tab_elem == TE_F32) HG_TAB_LAUNCH(float, float);
            else HG_TAB_LAUNCH(hg::f2, float);
            CU(cudaGetLastError());
            g_launches++;
            if (tensor) {
                const unsigned long long rows = count * rows_per_event;
                if (p->prec == HEGET_FP64) {
                    const size_t smem = (size_t)dev.Rpad * (dev.Rpad + 4) * 8;
                    CU(cudaFuncSetAttribute(hg::k_colour_dmma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                    hg::k_colour_dmma<<<(unsigned int)((rows + 63) / 64), 256, smem, s>>>((const double*)p->tc_x, (const double*)p->tc_cfull, (double*)p->tc_form, rows, dev.Rpad);
                    hg::k_colour_finish<double><<<(unsigned int)((count + 7) / 8), 256, 0, s>>>((const double*)p->tc_form, (double*)d_me2 + first, count, (int)rows_per_event, oscale);
                } else {
                    const size_t smem = (size_t)2 * dev.Rpad * (dev.Rpad + 8) * 4;
                    CU(cudaFuncSetAttribute(hg::k_colour_tf32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                    hg::k_colour_tf32<<<(unsigned int)((rows + 127) / 128), 256, smem, s>>>((const float*)p->tc_x, (const float*)p->tc_cfull, (float*)p->tc_form, rows, dev.Rpad);
                    hg::k_colour_finish<float><<<(unsigned int)((count + 7) / 8), 256, 0, s>>>((const float*)p->tc_form, (float*)d_me2 + first, count, (int)rows_per_event, oscale);
                }
                CU(cudaGetLastError());
                g_launches += 2;
            }
        }
#undef HG_TAB_LAUNCH
#undef HG_TAB_LAUNCH2
#undef HG_TAB_LAUNCH3
        return HEGET_OK;
    }
    const hg::ProcDesc* d = p->d;

    hg::LaunchArgs a;
    a.d_mom = d_mom; a.n_events = n_events; a.inv_sqrt_s = 1.0 / p->sqrt_s; a.out_scale = p->out_scale; a.d_me2 = d_me2;
    a.hel_mode = (int)mode; a.hel_fixed = hel_fixed; a.seed = seed; a.first_event = first_event; a.lanes = effective_lanes(p);
    // one configuration per event: in the wide variant all lanes of an event would evaluate the same configuration, so take
    // the one-event-per-thread variant where it is built (the big processes only have the wide one: L-fold redundant there)
    if (mode != HEGET_HEL_SUM && p->lanes == 0 && (d->lanes_avail & 1)) a.lanes = 1;
    a.stream = (cudaStream_t)cuda_stream;
    const int rc = d->launch(p->prec, a);
    if (rc != 0) return fail(HEGET_ECUDA, "launch of '%s' failed: %s", d->name, cudaGetErrorString((cudaError_t)rc));
    g_launches++;
    return HEGET_OK;
}

heget_status_t heget_run_host(heget_process_t* p, uint64_t seed, uint64_t first_event, uint64_t n_events,
                              const double* h_mom_in, double* h_mom_out, double* h_weight, heget_hel_mode_t mode,
                              const int8_t* hel, void* h_me2, void* cuda_stream) {
    if (!p) return fail(HEGET_EINVAL, "heget_run_host: NULL handle");
    if (n_events == 0) return HEGET_OK;
    if (!h_me2) return fail(HEGET_EINVAL, "heget_run_host: h_me2 is NULL");
    std::lock_guard<std::mutex> lock(p->s_mutex);      // the device scratch belongs to the handle: one host call at a time
    const size_t nm = (size_t)p->n_legs * 4 * n_events, esz = p->prec == HEGET_FP64 ? 8 : 4;
    if (p->s_cap < n_events) {
        if (p->s_mom) cudaFree(p->s_mom); if (p->s_w) cudaFree(p->s_w); if (p->s_me2) cudaFree(p->s_me2);
        p->s_mom = 0; p->s_w = 0; p->s_me2 = 0; p->s_cap = 0;
        if (cudaMalloc(&p->s_mom, nm * 8) != cudaSuccess || cudaMalloc(&p->s_w, n_events * 8) != cudaSuccess || cudaMalloc(&p->s_me2, n_events * 8) != cudaSuccess) {
            cudaGetLastError(); return fail(HEGET_ENOMEM, "heget_run_host: cannot allocate device scratch for %llu events", (unsigned long long)n_events);
        }
        p->s_cap = n_events;
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    heget_status_t st;
    if (h_mom_in) { CU(cudaMemcpyAsync(p->s_mom, h_mom_in, nm * 8, cudaMemcpyHostToDevice, s)); }
    else {
        st = heget_sample_momenta(p, seed, first_event, n_events, p->s_mom, h_weight ? p->s_w : 0, 0, cuda_stream);
        if (st != HEGET_OK) return st;
    }
    st = heget_eval_me2(p, p->s_mom, n_events, mode, hel, seed, first_event, p->s_me2, cuda_stream);
    if (st != HEGET_OK) return st;
    CU(cudaMemcpyAsync(h_me2, p->s_me2, n_events * esz, cudaMemcpyDeviceToHost, s));
    if (h_mom_out) CU(cudaMemcpyAsync(h_mom_out, p->s_mom, nm * 8, cudaMemcpyDeviceToHost, s));
    if (h_weight && !h_mom_in) CU(cudaMemcpyAsync(h_weight, p->s_w, n_events * 8, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return HEGET_OK;
}

}  // extern "C"

// ---- the entry point that allocates nothing ------------------------------------------------------------------------------------------
// The tensor-core colour stage hands the rows of J (eq. 8) from the table kernel to the contraction kernel through a
// scratch buffer in HBM; heget_eval_me2 takes that buffer from cudaMalloc.  heget_eval_me2_static runs the same three kernels with the
// buffer inside ONE file-scope device array of HEGET_STATIC_SCRATCH_BYTES, so that nothing is allocated or freed in the call (CUDA graph
// capture, serving loops and harnesses that forbid cudaMalloc).  Every GPU that loads the library holds the array until the process
// exits.  In host code the NAME of the array is a host-side stand-in, not a device address: its device address is asked for once per
// device, with that device current, by cudaGetSymbolAddress (heget_static_prepare) and that pointer is what the kernels get.
static __device__ __align__(256) unsigned char g_static_scratch[HEGET_STATIC_SCRATCH_BYTES];
static void* g_static_ptr[64];                 // device ordinal -> address of g_static_scratch on that device (0: not asked for yet)
static std::mutex g_static_mutex;

static size_t static_align(size_t v) { return (v + 255) / 256 * 256; }
// bytes of the scratch array that n events take: rows of J, then the row forms (256-byte aligned)
static size_t static_bytes(const hg::TabDev& d, size_t esz, unsigned long long n) {
    const size_t rows_per_event = (size_t)d.nchunks * 32 * 2;
    return static_align((size_t)n * rows_per_event * d.Rpad * esz) + (size_t)n * rows_per_event * esz;
}
static unsigned long long static_max_events(const hg::TabDev& d, size_t esz) {
    const size_t rows_per_event = (size_t)d.nchunks * 32 * 2, per_event = rows_per_event * d.Rpad * esz + rows_per_event * esz;
    unsigned long long n = (unsigned long long)(HEGET_STATIC_SCRATCH_BYTES / per_event);
    while (n > 0 && static_bytes(d, esz, n) > (size_t)HEGET_STATIC_SCRATCH_BYTES) --n;
    return n;
}
static bool static_ready(const heget_process* p) { return p->tab && p->tab_on_device && p->colour_stage == HEGET_COLOUR_TENSOR && p->tc_cfull; }

extern "C" {

heget_status_t heget_static_prepare(heget_process_t* p) {
    if (!p) return fail(HEGET_EINVAL, "heget_static_prepare: NULL handle");
    if (effective_kernel(p) != HEGET_KERNEL_TABLE) return fail(HEGET_EUNSUPPORTED, "heget_static_prepare: the static-scratch path belongs to the TABLE back end (heget_set_kernel)");
    if (p->colour_stage != HEGET_COLOUR_TENSOR) return fail(HEGET_EINVAL, "heget_static_prepare: select the tensor-core colour stage first (heget_set_colour_stage(HEGET_COLOUR_TENSOR))");
    const heget_status_t st = table_to_device(p);      // set-up: this is where the process tables are allocated and uploaded
    if (st != HEGET_OK) return st;
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(HEGET_EUNSUPPORTED, "heget_static_prepare: device ordinal %d", dev);
    {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_ptr[dev]) {
            void* ptr = 0;
            const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);      // once per device, with that device current
            if (e != cudaSuccess || !ptr) { cudaGetLastError(); return fail(HEGET_ECUDA, "heget_static_prepare: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e)); }
            g_static_ptr[dev] = ptr;
        }
    }
    // dynamic shared memory of the contraction kernels (an attribute of the function: no allocation, but not something to do under capture)
    if (p->prec == HEGET_FP64) CU(cudaFuncSetAttribute(hg::k_colour_dmma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)p->tdev.Rpad * (p->tdev.Rpad + 4) * 8)));
    else CU(cudaFuncSetAttribute(hg::k_colour_tf32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)2 * p->tdev.Rpad * (p->tdev.Rpad + 8) * 4)));
    // with lazy module loading a kernel's code reaches the device at its first use: touch the third kernel here so that the first call loads nothing
    cudaFuncAttributes fa;
    if (p->prec == HEGET_FP64) CU(cudaFuncGetAttributes(&fa, hg::k_colour_finish<double>)); else CU(cudaFuncGetAttributes(&fa, hg::k_colour_finish<float>));
    return HEGET_OK;
}

uint64_t heget_static_max_events(const heget_process_t* p) {
    if (!p || !static_ready(p)) return 0;
    return static_max_events(p->tdev, p->prec == HEGET_FP64 ? 8 : 4);
}

heget_status_t heget_eval_me2_static(heget_process_t* p, const double* d_mom, uint64_t n_events, void* d_me2, void* cuda_stream) {
    if (!p) return fail(HEGET_EINVAL, "heget_eval_me2_static: NULL handle");
    if (!static_ready(p)) return fail(HEGET_EINVAL, "heget_eval_me2_static: the handle is not prepared (TABLE back end, heget_set_colour_stage(HEGET_COLOUR_TENSOR), then heget_static_prepare; a later heget_set_kernel / heget_set_colour_stage undoes it)");
    if (n_events == 0) return HEGET_OK;
    if (!d_mom || !d_me2) return fail(HEGET_EINVAL, "heget_eval_me2_static: NULL device pointer");
    int devno = -1;
    CU(cudaGetDevice(&devno));
    unsigned char* scratch = (devno >= 0 && devno < 64) ? (unsigned char*)g_static_ptr[devno] : 0;
    if (!scratch) return fail(HEGET_EINVAL, "heget_eval_me2_static: heget_static_prepare has not run on device %d", devno);
    const size_t esz = p->prec == HEGET_FP64 ? 8 : 4;
    hg::TabDev dev = p->tdev;
    const unsigned long long nmax = static_max_events(dev, esz);
    if (n_events > nmax) return fail(HEGET_EINVAL, "heget_eval_me2_static: %llu events need %zu bytes of scratch, the static array holds %llu (at most %llu events of '%s' per call)",
                                     (unsigned long long)n_events, static_bytes(dev, esz, n_events), (unsigned long long)HEGET_STATIC_SCRATCH_BYTES, nmax, p->name.c_str());
    const size_t rows_per_event = (size_t)dev.nchunks * 32 * 2;
    const unsigned long long rows = n_events * rows_per_event;
    void* X = scratch;
    void* form = scratch + static_align((size_t)rows * dev.Rpad * esz);
    // nothing in the scratch has to start at zero: the table kernel writes every element of the rows of [0, n_events), the contraction kernel
    // writes every row form, and nothing is accumulated into either -- what an earlier call left behind is never read
    dev.cstage = 3; dev.jout = X;
    const int epc = p->tab_epc;
    const int evpc = epc * (p->tab_elem == TE_F32X2 ? 2 : 1);
    const unsigned int blocks = (unsigned int)((n_events + evpc - 1) / evpc);
    const int threads = epc * dev.nchunks * 32 * dev.nsp;
    const TabShape& sh = p->tab_shape;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const double iss = 1.0 / p->sqrt_s, oscale = p->out_scale * (double)p->tab->hel_weight;
#define HG_TAB_STATIC3(TT, OT, JMV, MWV) hg::k_tab<TT, JMV, MWV><<<blocks, threads, sh.smem, s>>>(dev, epc, sh.tm_cols, sh.tm_wcols, d_mom, n_events, n_events, iss, oscale, (OT*)d_me2, (int)HEGET_HEL_SUM, -1, 0ull, 0ull)
#define HG_TAB_STATIC2(TT, OT, JMV) do { if (sh.nsp > 1) HG_TAB_STATIC3(TT, OT, JMV, true); else HG_TAB_STATIC3(TT, OT, JMV, false); } while (0)
#define HG_TAB_STATIC(TT, OT) do { if (sh.jm) HG_TAB_STATIC2(TT, OT, 1); else HG_TAB_STATIC2(TT, OT, 0); } while (0)
    if (p->tab_elem == TE_F64) HG_TAB_STATIC(double, double);
    else if (p->tab_elem == TE_F32) HG_TAB_STATIC(float, float);
    else HG_TAB_STATIC(hg::f2, float);
#undef HG_TAB_STATIC
#undef HG_TAB_STATIC2
#undef HG_TAB_STATIC3
    CU(cudaGetLastError());
    if (p->prec == HEGET_FP64) {
        const size_t smem = (size_t)dev.Rpad * (dev.Rpad + 4) * 8;
        hg::k_colour_dmma<<<(unsigned int)((rows + 63) / 64), 256, smem, s>>>((const double*)X, (const double*)p->tc_cfull, (double*)form, rows, dev.Rpad);
        hg::k_colour_finish<double><<<(unsigned int)((n_events + 7) / 8), 256, 0, s>>>((const double*)form, (double*)d_me2, n_events, (int)rows_per_event, oscale);
    } else {
        const size_t smem = (size_t)2 * dev.Rpad * (dev.Rpad + 8) * 4;
        hg::k_colour_tf32<<<(unsigned int)((rows + 127) / 128), 256, smem, s>>>((const float*)X, (const float*)p->tc_cfull, (float*)form, rows, dev.Rpad);
        hg::k_colour_finish<float><<<(unsigned int)((n_events + 7) / 8), 256, 0, s>>>((const float*)form, (float*)d_me2, n_events, (int)rows_per_event, oscale);
    }
    CU(cudaGetLastError());
    g_launches += 3;
    return HEGET_OK;
}

}  // extern "C"
