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
#include <string>
#include <vector>
#include <dlfcn.h>
#include <sys/stat.h>
#include <unistd.h>
#include "../../include/heget.h"
#include "rambo.cuh"

extern "C" int heget_generate_source(const char* tag, const char* process, const char* out_path, char* msg, int msglen);

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

heget_status_t open_plugin(const std::string& so, const std::string& key, const hg::ProcDesc** out) {
    void* h = dlopen(so.c_str(), RTLD_NOW | RTLD_LOCAL);
    if (!h) return fail(HEGET_ECOMPILE, "dlopen %s: %s", so.c_str(), dlerror());
    typedef const hg::ProcDesc* (*fn_t)();
    fn_t fn = (fn_t)dlsym(h, "heget_plugin_desc");
    if (!fn) return fail(HEGET_ECOMPILE, "%s exports no heget_plugin_desc", so.c_str());
    *out = g_plugins[key] = fn();
    return HEGET_OK;
}

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
    if (exists(dir + "/heget_" + key + ".so")) return open_plugin(dir + "/heget_" + key + ".so", key, out);
    const std::string dst = wdir + "/heget_" + key + ".so";
    if (exists(dst)) return open_plugin(dst, key, out);
    mkdir(wdir.c_str(), 0755);
    const std::string cu = wdir + "/gen_" + tag + ".cu", log = wdir + "/gen_" + key + ".log", tmp = dst + ".tmp";
    char msg[512] = "";
    const int rc = heget_generate_source(tag.c_str(), name.c_str(), cu.c_str(), msg, sizeof msg);
    if (rc == 1) return fail(HEGET_EINVAL, "process '%s': %s", name.c_str(), msg);
    if (rc == 2) return fail(HEGET_EUNSUPPORTED, "process '%s': %s", name.c_str(), msg);
    if (rc != 0) return fail(HEGET_ECOMPILE, "generator failed for '%s': %s", name.c_str(), msg);
    const char* nvcc = getenv("HEGET_NVCC");
    const std::string cmd = std::string(nvcc ? nvcc : "nvcc") + " -std=c++17 -O3 -gencode arch=compute_100a,code=sm_100a -lineinfo -shared -Xcompiler -fPIC" +
                            " -DHG_ONLY_PREC=" + (prec == 0 ? "0" : prec == 1 ? "1" : "2") + (n_legs >= 6 ? " -DHG_NO_LANES1" : "") + " -I'" + lib_dir() + "/csrc/device' -o '" + tmp +
                            "' '" + cu + "' > '" + log + "' 2>&1";
    if (system(cmd.c_str()) != 0) return fail(HEGET_ECOMPILE, "nvcc failed for '%s' (see %s)", name.c_str(), log.c_str());
    if (rename(tmp.c_str(), dst.c_str()) != 0) return fail(HEGET_ECOMPILE, "cannot install %s", dst.c_str());
    return open_plugin(dst, key, out);
}

double rambo_flat_weight(int n, double sqrt_s) {      // reading A7: (pi/2)^(n-1) s^(n-2) / ((n-1)!(n-2)!) (2 pi)^(4-3n)
    const double PI = 3.14159265358979323846;
    double w = pow(PI / 2.0, n - 1) * pow(sqrt_s * sqrt_s, n - 2) * pow(2.0 * PI, 4 - 3 * n);
    for (int k = 2; k <= n - 1; ++k) w /= (double)k;
    for (int k = 2; k <= n - 2; ++k) w /= (double)k;
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

struct heget_process;
static int effective_lanes(const heget_process* p);

struct heget_process {
    const hg::ProcDesc* d;
    int prec, lanes;
    double sqrt_s, alpha_s, out_scale;
    heget_cuts_t cuts;
    // scratch of the host-buffer entry point
    double* s_mom; double* s_w; void* s_me2; size_t s_cap;
};

// lanes = 0 (automatic): FP64 takes the wide variant (event-cache reads become warp broadcasts; measured 26 vs 23 TFLOP/s on
// C2), FP32 the one-event-per-thread variant where it is built (the compiler keeps the event cache in registers across the
// helicity loop; measured 53 vs 40 TFLOP/s on C2)
static int effective_lanes(const heget_process* p) {
    if (p->lanes) return p->lanes;
    return (p->prec == HEGET_FP32 && (p->d->lanes_avail & 1)) ? 1 : p->d->lanes_wide;
}

extern "C" {

const char* heget_last_error(void) { return g_err; }
uint64_t heget_launch_count(void) { return g_launches.load(); }

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
    const hg::ProcDesc* d = 0;
    heget_status_t st = load_plugin(name, tag, n_legs, (int)prec, &d);
    if (st != HEGET_OK) return st;
    heget_process* p = new (std::nothrow) heget_process();
    if (!p) return fail(HEGET_ENOMEM, "out of host memory");
    p->d = d; p->prec = (int)prec; p->lanes = 0; p->sqrt_s = sqrt_s_hat; p->alpha_s = alpha_s;
    p->cuts.pt_min = cuts ? cuts->pt_min : 0.0; p->cuts.eta_max = cuts ? cuts->eta_max : 0.0; p->cuts.dr_min = cuts ? cuts->dr_min : 0.0;
    // S * 1/4 * 1/(n_a n_b) * g_s^(2(n-2)) * s_hat^-(n-4): the kernels work in units of sqrt(s_hat) (reading A21)
    const double gs2 = 4.0 * 3.14159265358979323846 * alpha_s;
    p->out_scale = d->sym_factor * d->avg_spin * d->avg_color * pow(gs2, d->n_ext - 2) * pow(sqrt_s_hat, -2.0 * (d->n_ext - 4));
    p->s_mom = 0; p->s_w = 0; p->s_me2 = 0; p->s_cap = 0;
    *out = p;
    return HEGET_OK;
}

void heget_destroy(heget_process_t* p) {
    if (!p) return;
    if (p->s_mom) cudaFree(p->s_mom);
    if (p->s_w) cudaFree(p->s_w);
    if (p->s_me2) cudaFree(p->s_me2);
    delete p;
}

heget_status_t heget_set_lanes(heget_process_t* p, int lanes) {
    if (!p) return fail(HEGET_EINVAL, "heget_set_lanes: NULL handle");
    const hg::ProcDesc* d = p->d;
    const bool ok = lanes == 0 || (lanes == 1 && (d->lanes_avail & 1)) || (lanes == d->lanes_wide && (d->lanes_avail & 2));
    if (!ok) return fail(HEGET_EINVAL, "heget_set_lanes: lanes = %d is not built for '%s' (0 = automatic%s, wide = %d)", lanes, d->name,
                         (d->lanes_avail & 1) ? ", 1" : "", d->lanes_wide);
    p->lanes = lanes; return HEGET_OK;
}

heget_status_t heget_process_info(const heget_process_t* p, heget_info_t* o) {
    if (!p || !o) return fail(HEGET_EINVAL, "heget_process_info: NULL argument");
    const hg::ProcDesc* d = p->d;
    memset(o, 0, sizeof *o);
    o->n_ext = d->n_ext; o->n_hel = d->n_hel; o->n_hel_eval = d->n_hel_eval; o->n_diagrams = d->n_diagrams; o->n_topologies = d->n_topologies;
    o->n_color = d->n_color; o->n_color_eval = d->n_color_eval; o->n_color_reduced = d->n_color_reduced;
    o->avg_spin = d->avg_spin; o->avg_color = d->avg_color; o->sym_factor = d->sym_factor;
    o->flops_per_event = d->flops_per_event; o->flops_per_helicity = d->flops_per_hel;
    o->threads_per_block = d->block[p->prec == HEGET_FP32 ? 1 : 0]; o->lanes_wide = d->lanes_wide; o->lanes = effective_lanes(p);
    o->regs_per_thread = -1; o->local_bytes_per_thread = -1;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0) {
        hg::KernelInfo ki;
        if (d->kernel_info(p->prec, effective_lanes(p), &ki) == 0) { o->regs_per_thread = ki.regs; o->local_bytes_per_thread = ki.local_bytes; o->threads_per_block = ki.block; }
        else cudaGetLastError();
    } else cudaGetLastError();
    return HEGET_OK;
}

heget_status_t heget_color_matrix(const heget_process_t* p, int which, double* h_out, int* n) {
    if (!p || !n) return fail(HEGET_EINVAL, "heget_color_matrix: NULL argument");
    if (which != 0 && which != 1) return fail(HEGET_EINVAL, "heget_color_matrix: which must be 0 or 1");
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
    const int nf = p->d->n_ext - 2;
    hg::RamboArgs a;
    a.sqrt_s = p->sqrt_s; a.pt_min = p->cuts.pt_min; a.eta_max = p->cuts.eta_max; a.dr_min = p->cuts.dr_min;
    a.w0 = rambo_flat_weight(nf, p->sqrt_s);
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
    const hg::ProcDesc* d = p->d;
    hg::LaunchArgs a;
    a.d_mom = d_mom; a.n_events = n_events; a.inv_sqrt_s = 1.0 / p->sqrt_s; a.out_scale = p->out_scale; a.d_me2 = d_me2;
    a.hel_mode = (int)mode; a.hel_fixed = -1; a.seed = seed; a.first_event = first_event; a.d_jbuf = 0; a.lanes = effective_lanes(p);
    // one configuration per event: in the wide variant all lanes of an event would evaluate the same configuration, so take
    // the one-event-per-thread variant where it is built (the big processes only have the wide one: L-fold redundant there)
    if (mode != HEGET_HEL_SUM && p->lanes == 0 && (d->lanes_avail & 1)) a.lanes = 1;
    a.stream = (cudaStream_t)cuda_stream;
    if (mode == HEGET_HEL_FIXED) {
        for (int i = 0; i < d->n_ext; ++i) if (hel[i] != 1 && hel[i] != -1) return fail(HEGET_EINVAL, "heget_eval_me2: hel[%d] = %d is not +-1", i, (int)hel[i]);
        for (int h = 0; h < d->n_hel_eval && a.hel_fixed < 0; ++h) {
            bool same = true;
            for (int i = 0; i < d->n_ext; ++i) if (d->hel_table[h * d->n_ext + i] != hel[i]) { same = false; break; }
            if (same) a.hel_fixed = h;
        }
    }
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
    const size_t nm = (size_t)p->d->n_ext * 4 * n_events, esz = p->prec == HEGET_FP64 ? 8 : 4;
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
