// rt_api.cu — the C ABI of include/rt.h: argument validation, the handle, kernel launches.
// No physics here: every step of the path runs in the kernels of rt_kernels_*.cuh.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "../../include/rt.h"
#include "rt_kernels_fused.cuh"
#include "rt_kernels_measure.cuh"
#include "rt_fused_inst.cuh"

// k_substep_fused is instantiated in rt_fused_inst.cu (several translation units, compiled side by side)
namespace rtm1 {
#define RT_EXTERN(P, A, B, C_, D_, E_, F_, G_)                                                                                    \
    extern template __global__ void k_substep_fused<A, B, C_, D_, E_, F_, G_>(const __grid_constant__ GridDev, const __grid_constant__ ParamsDev, const __grid_constant__ OpacDev, \
        const __grid_constant__ OpacDev, const __grid_constant__ OpacDev, const __grid_constant__ FusedArgs, const __grid_constant__ FusedMaps, int);
RT_FUSED_INSTANCES(RT_EXTERN)
#undef RT_EXTERN
}  // namespace rtm1

using namespace rtm1;

struct rt_grid {
    GridDev dev;
    cudaStream_t stream;
    int device;                 // the device the handle was created on (every entry point switches to it)
    double* metric_buf;
    double* lim;  // thick-limit pre-pass array, ntot doubles (lazily allocated)
    double* rk_save[4];  // rt_rk2_step: T^n, m^n (lazily allocated)
    double* rk_dt;       // rt_rk2_step: the dt each stage reads (and overwrites)
    const double* divfirr;  // rt_set_irradiation: caller-owned device array or nullptr
    int face_fix;  // rt_set_face_fix: RT_FIX_*
    int recon;     // rt_set_reconstruction: RT_RECON_*
    double limo3_r;
    double* kpr;  // rho kappa_P per cell, written by the pre-pass of the fused sub-step (lazily allocated)
    CflScratch* scr;
    double* dt_dev;
    double* dt_pinned;
    unsigned long long* counters;  // device: floor, clip
    unsigned long long* counters_pinned;
    rt_params par;
    int have_par;
    OpacDev opac[3];
    double* table_dev[3];
    std::vector<double> table_host[3];
    rt_opacity opac_host[3];
    int same_PR;
    int march_len;
    int fused_tma_off;  // test hook (env RT_M1_NO_TMA at grid creation): stage the planes by cp.async even where TMA could
    int fused_seg;  // rt_set_tuning: 0 auto, -1 never use the fused sub-step kernel, > 0 its x3 segment length
    long long launches;
    // TMA descriptors of the fused kernel, keyed by the five staged arrays: rt_substep alternates between two buffer
    // sets, so a handful of entries serves a whole run without re-encoding (the grid shape never changes)
    struct MapEntry { const double* key[FNARR]; int narr; FusedMaps maps; };
    std::vector<MapEntry> map_cache;
    // optional per-kernel device timing (rt_set_profiling): one event pair per launch
    int profiling;
    struct ProfRec { int kind; cudaEvent_t a, b; };
    std::vector<ProfRec> prof;
    double prof_ms[RT_NKERNEL_KINDS];     // sums already folded in by ProfScope::trim
    long long prof_n[RT_NKERNEL_KINDS];
    char err[256];
};

// RAII around one launch: records an event before and after it when profiling is on
struct ProfScope {
    rt_grid* g;
    cudaStream_t st;
    cudaEvent_t b;
    ProfScope(rt_grid* g_, int kind, cudaStream_t st_ = nullptr) : g(g_), st(st_ ? st_ : g_->stream), b(nullptr) {
        if (!g->profiling) return;
        cudaEvent_t a = nullptr;
        if (cudaEventCreate(&a) != cudaSuccess) return;
        if (cudaEventCreate(&b) != cudaSuccess) {
            cudaEventDestroy(a);
            b = nullptr;
            return;
        }
        cudaEventRecord(a, st);
        g->prof.push_back({kind, a, b});
    }
    // called by the launch sites BEFORE a new scope opens: with too many pairs outstanding, fold the finished ones into the
    // running sums (synchronises the stream once per kMaxLive launches) so that a long profiled run holds a bounded number
    static void trim(rt_grid* g) {
        constexpr size_t kMaxLive = 4096;
        if (!g->profiling || g->prof.size() < kMaxLive) return;
        if (cudaStreamSynchronize(g->stream) != cudaSuccess) return;
        for (auto& r : g->prof) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess && r.kind >= 0 && r.kind < RT_NKERNEL_KINDS) {
                g->prof_ms[r.kind] += (double)t;
                g->prof_n[r.kind] += 1;
            }
            cudaEventDestroy(r.a);
            cudaEventDestroy(r.b);
        }
        g->prof.clear();
    }
    ~ProfScope() {
        if (b) cudaEventRecord(b, st);
    }
};

// Every entry point runs on the device the handle was created on, whatever the caller's current device is, and
// restores the caller's device on the way out.
struct DeviceGuard {
    int prev;
    bool switched;
    explicit DeviceGuard(const rt_grid* g) : prev(-1), switched(false) {
        if (!g) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != g->device) switched = cudaSetDevice(g->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

static int32_t fail(rt_grid* g, int32_t code, const char* fmt, ...) {
    if (g) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(g->err, sizeof(g->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define RT_CUDA(g, call)                                                                                       \
    do {                                                                                                       \
        cudaError_t e_ = (call);                                                                               \
        if (e_ != cudaSuccess) return fail((g), RT_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_));      \
    } while (0)

#define RT_LAUNCH_CHECK(g)                                                                                     \
    do {                                                                                                       \
        (g)->launches += 1;                                                                                    \
        cudaError_t e_ = cudaGetLastError();                                                                   \
        if (e_ != cudaSuccess) return fail((g), RT_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(e_));    \
    } while (0)

static bool aligned8(const void* p) { return p && (reinterpret_cast<uintptr_t>(p) & 7u) == 0; }

extern "C" const char* rt_last_error(const rt_grid* g) { return g ? g->err : "null grid handle"; }
extern "C" int64_t rt_get_launch_count(const rt_grid* g) {
    DeviceGuard dg_(g); return g ? g->launches : 0; }

extern "C" int32_t rt_set_profiling(rt_grid* g, int32_t on) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    g->profiling = on ? 1 : 0;
    return RT_OK;
}

extern "C" int32_t rt_get_kernel_times(rt_grid* g, double ms[RT_NKERNEL_KINDS], int64_t launches[RT_NKERNEL_KINDS]) {
    DeviceGuard dg_(g);
    if (!g || !ms || !launches) return fail(g, RT_ERR_INVALID_ARG, "rt_get_kernel_times: null argument");
    for (int k = 0; k < RT_NKERNEL_KINDS; ++k) {
        ms[k] = g->prof_ms[k];
        launches[k] = g->prof_n[k];
        g->prof_ms[k] = 0.0;
        g->prof_n[k] = 0;
    }
    RT_CUDA(g, cudaStreamSynchronize(g->stream));
    for (auto& r : g->prof) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess && r.kind >= 0 && r.kind < RT_NKERNEL_KINDS) {
            ms[r.kind] += (double)t;
            launches[r.kind] += 1;
        }
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    g->prof.clear();
    return RT_OK;
}

extern "C" int32_t rt_set_tuning(rt_grid* g, int32_t march_len, int32_t fused_seg) {
    DeviceGuard dg_(g);
    if (!g || march_len < 0 || fused_seg < -1) return fail(g, RT_ERR_INVALID_ARG, "rt_set_tuning: bad argument");
    g->march_len = march_len;
    g->fused_seg = fused_seg;
    return RT_OK;
}

// ------------------------------------------------------------------------------------------------
extern "C" int32_t rt_grid_create(int32_t geometry, const int32_t n[3], int32_t nghost, const double* x1f,
                                  const double* x2f, const double* x3f, const int32_t bc[6], void* cuda_stream,
                                  rt_grid** out) {
    if (!n || !x1f || !x2f || !x3f || !bc || !out) return RT_ERR_INVALID_ARG;
    *out = nullptr;
    if (geometry < 0 || geometry > 2 || nghost != 2) return RT_ERR_INVALID_ARG;
    const double* xf[3] = {x1f, x2f, x3f};
    for (int d = 0; d < 3; ++d) {
        if (n[d] < 1 || n[d] > (1 << 24)) return RT_ERR_INVALID_ARG;
        for (int i = 0; i <= n[d]; ++i)
            if (!isfinite(xf[d][i])) return RT_ERR_INVALID_ARG;
        for (int i = 0; i < n[d]; ++i)
            if (!(xf[d][i + 1] > xf[d][i])) return RT_ERR_INVALID_ARG;
        if (bc[2 * d] < 0 || bc[2 * d] > 3 || bc[2 * d + 1] < 0 || bc[2 * d + 1] > 3) return RT_ERR_INVALID_ARG;
        if ((bc[2 * d] == RT_BC_PERIODIC) != (bc[2 * d + 1] == RT_BC_PERIODIC)) return RT_ERR_INVALID_ARG;
    }
    if (geometry != RT_CARTESIAN && x1f[0] < 0.0) return RT_ERR_INVALID_ARG;
    if (geometry == RT_SPHERICAL && (x2f[0] < 0.0 || x2f[n[1]] > M_PI)) return RT_ERR_INVALID_ARG;
    // the geometric sources ride on the x1 sweep: curvilinear grids need an active x1
    if (geometry != RT_CARTESIAN && n[0] < 2) return RT_ERR_INVALID_ARG;
    // x2 / x3 indices ride in gridDim.y / gridDim.z of several launches (limit 65535)
    if (n[1] > 65535 || n[2] > 65535) return RT_ERR_INVALID_ARG;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return RT_ERR_CUDA;  // no CPU fallback

    rt_grid* g = new (std::nothrow) rt_grid();
    if (!g) return RT_ERR_CUDA;
    memset(&g->dev, 0, sizeof(g->dev));
    g->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    g->device = 0;
    cudaGetDevice(&g->device);
    g->metric_buf = nullptr;
    g->lim = nullptr;
    g->kpr = nullptr;
    g->divfirr = nullptr;
    g->face_fix = RT_FIX_FPRESERVING;
    g->recon = RT_RECON_PLM;
    g->limo3_r = 0.0;
    for (int q = 0; q < 4; ++q) g->rk_save[q] = nullptr;
    g->rk_dt = nullptr;
    g->scr = nullptr;
    g->dt_dev = nullptr;
    g->dt_pinned = nullptr;
    g->counters = nullptr;
    g->counters_pinned = nullptr;
    g->have_par = 0;
    g->same_PR = 0;
    g->march_len = 0;
    g->fused_seg = 0;
    {
        const char* e = getenv("RT_M1_NO_TMA");
        g->fused_tma_off = (e && e[0] == '1') ? 1 : 0;
    }
    g->launches = 0;
    g->profiling = 0;
    for (int k = 0; k < RT_NKERNEL_KINDS; ++k) {
        g->prof_ms[k] = 0.0;
        g->prof_n[k] = 0;
    }
    g->err[0] = 0;
    for (int w = 0; w < 3; ++w) {
        memset(&g->opac[w], 0, sizeof(OpacDev));
        memset(&g->opac_host[w], 0, sizeof(rt_opacity));
        g->table_dev[w] = nullptr;
    }
    GridDev& D = g->dev;
    D.geometry = geometry;
    for (int d = 0; d < 3; ++d) {
        D.n[d] = n[d];
        D.gh[d] = n[d] > 1 ? nghost : 0;
        D.nt[d] = n[d] + 2 * D.gh[d];
        D.bc[2 * d] = bc[2 * d];
        D.bc[2 * d + 1] = bc[2 * d + 1];
    }
    D.stride[0] = 1;
    D.stride[1] = D.nt[0];
    D.stride[2] = (long long)D.nt[0] * D.nt[1];
    D.ntot = D.stride[2] * D.nt[2];

    // one device buffer for edges and every 1-D factor array: per axis e,
    //   xf (n+1), wf (n+1), vf (n), and 4 x 3 arrays (af, cg, len, ilen)[d][e] of n; plus invr (n1), cot (n2)
    size_t total = 0;
    for (int e = 0; e < 3; ++e) total += 2 * (size_t)(n[e] + 1) + (size_t)n[e] * (1 + 12);
    total += (size_t)n[0] + (size_t)n[1];
    cudaError_t ce = cudaMalloc(&g->metric_buf, total * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc(&g->scr, sizeof(CflScratch));
    if (ce == cudaSuccess) ce = cudaMalloc(&g->dt_dev, sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc(&g->counters, 2 * sizeof(unsigned long long));
    if (ce == cudaSuccess) ce = cudaMallocHost(&g->dt_pinned, sizeof(double));
    if (ce == cudaSuccess) ce = cudaMallocHost(&g->counters_pinned, 2 * sizeof(unsigned long long));
    if (ce == cudaSuccess) ce = cudaMemsetAsync(g->scr, 0, sizeof(CflScratch), g->stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(g->counters, 0, 2 * sizeof(unsigned long long), g->stream);
    if (ce != cudaSuccess) {
        rt_grid_destroy(g);
        return RT_ERR_CUDA;
    }
    MetricOut M;
    double* p = g->metric_buf;
    double* xdev[3];
    for (int e = 0; e < 3; ++e) {
        xdev[e] = p; D.xf[e] = p; p += n[e] + 1;
        M.wf[e] = p; D.wf[e] = p; p += n[e] + 1;
        M.vf[e] = p; D.vf[e] = p; p += n[e];
    }
    for (int d = 0; d < 3; ++d)
        for (int e = 0; e < 3; ++e) {
            M.af[d][e] = p; D.af[d][e] = p; p += n[e];
            M.cg[d][e] = p; D.cg[d][e] = p; p += n[e];
            M.len[d][e] = p; D.len[d][e] = p; p += n[e];
            M.ilen[d][e] = p; D.ilen[d][e] = p; p += n[e];
        }
    M.invr = p; D.invr = p; p += n[0];
    M.cot = p; D.cot = p; p += n[1];
    for (int e = 0; e < 3 && ce == cudaSuccess; ++e)
        ce = cudaMemcpyAsync(xdev[e], xf[e], sizeof(double) * (size_t)(n[e] + 1), cudaMemcpyHostToDevice, g->stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(const_cast<double*>(D.invr), 0, sizeof(double) * (size_t)(n[0] + n[1]), g->stream);
    if (ce == cudaSuccess) {
        k_metric_precompute<<<8, 256, 0, g->stream>>>(D, M);
        g->launches += 1;
        ce = cudaGetLastError();
    }
    // host edge arrays may be freed by the caller on return: wait for the copies
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(g->stream);
    if (ce != cudaSuccess) {
        rt_grid_destroy(g);
        return RT_ERR_CUDA;
    }
    *out = g;
    return RT_OK;
}

extern "C" int32_t rt_grid_destroy(rt_grid* g) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    cudaStreamSynchronize(g->stream);
    for (auto& r : g->prof) {
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    cudaFree(g->metric_buf);
    cudaFree(g->lim);
    cudaFree(g->kpr);
    for (int q = 0; q < 4; ++q) cudaFree(g->rk_save[q]);
    cudaFree(g->rk_dt);
    cudaFree(g->scr);
    cudaFree(g->dt_dev);
    cudaFree(g->counters);
    cudaFreeHost(g->dt_pinned);
    cudaFreeHost(g->counters_pinned);
    for (int w = 0; w < 3; ++w) cudaFree(g->table_dev[w]);
    delete g;
    return RT_OK;
}

extern "C" int32_t rt_grid_get_metrics(rt_grid* g, double* vol, double* area1, double* area2, double* area3) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    const GridDev& D = g->dev;
    const size_t n1 = D.n[0], n2 = D.n[1], n3 = D.n[2];
    const size_t sz[4] = {n1 * n2 * n3, (n1 + 1) * n2 * n3, n1 * (n2 + 1) * n3, n1 * n2 * (n3 + 1)};
    double* host[4] = {vol, area1, area2, area3};
    double* dev[4] = {nullptr, nullptr, nullptr, nullptr};
    int32_t rc = RT_OK;
    for (int a = 0; a < 4 && rc == RT_OK; ++a)
        if (host[a] && cudaMalloc(&dev[a], sz[a] * sizeof(double)) != cudaSuccess) rc = fail(g, RT_ERR_CUDA, "cudaMalloc (metrics)");
    if (rc == RT_OK) {
        k_metric_expand<<<296, 256, 0, g->stream>>>(D, dev[0], dev[1], dev[2], dev[3]);
        g->launches += 1;
        if (cudaGetLastError() != cudaSuccess) rc = fail(g, RT_ERR_CUDA, "k_metric_expand launch failed");
    }
    for (int a = 0; a < 4 && rc == RT_OK; ++a)
        if (host[a] && cudaMemcpyAsync(host[a], dev[a], sz[a] * sizeof(double), cudaMemcpyDeviceToHost, g->stream) != cudaSuccess)
            rc = fail(g, RT_ERR_CUDA, "cudaMemcpyAsync (metrics)");
    if (cudaStreamSynchronize(g->stream) != cudaSuccess && rc == RT_OK) rc = fail(g, RT_ERR_CUDA, "stream sync (metrics)");
    for (int a = 0; a < 4; ++a) cudaFree(dev[a]);
    return rc;
}

extern "C" int32_t rt_set_params(rt_grid* g, const rt_params* p) {
    DeviceGuard dg_(g);
    if (!g || !p) return fail(g, RT_ERR_INVALID_ARG, "rt_set_params: null argument");
    if (!(p->chat > 0.0) || !(p->c > 0.0) || !(p->a_R >= 0.0) || !(p->c_v > 0.0) || !(p->E_floor >= 0.0) ||
        !isfinite(p->chat) || !isfinite(p->c) || !isfinite(p->a_R) || !isfinite(p->c_v) || !isfinite(p->E_floor))
        return fail(g, RT_ERR_INVALID_ARG, "rt_set_params: chat, c, c_v must be > 0 and a_R, E_floor >= 0");
    if (p->solver != RT_SOLVER_HLL && p->solver != RT_SOLVER_GLF && p->solver != RT_SOLVER_RUSANOV)
        return fail(g, RT_ERR_INVALID_ARG, "rt_set_params: unknown solver");
    g->par = *p;
    g->have_par = 1;
    return RT_OK;
}

static int half_int_exponent(double a) {
    const double t = 2.0 * a;
    if (t == rint(t) && fabs(t) <= 64.0) return (int)t;
    return INT_MIN;
}

static bool same_law(const rt_grid* g, int a, int b) {
    const rt_opacity &x = g->opac_host[a], &y = g->opac_host[b];
    if (!g->opac[a].set || !g->opac[b].set || x.kind != y.kind) return false;
    if (x.kind == 0)
        return x.kappa0 == y.kappa0 && x.rho0 == y.rho0 && x.T0 == y.T0 && x.a == y.a && x.b == y.b && x.kmin == y.kmin &&
               x.kmax == y.kmax;
    return x.n_lrho == y.n_lrho && x.n_lT == y.n_lT && x.lrho_min == y.lrho_min && x.lrho_max == y.lrho_max &&
           x.lT_min == y.lT_min && x.lT_max == y.lT_max && x.rho_unit == y.rho_unit && x.T_unit == y.T_unit &&
           g->table_host[a] == g->table_host[b];
}

extern "C" int32_t rt_set_opacity(rt_grid* g, int32_t which, const rt_opacity* o) {
    DeviceGuard dg_(g);
    if (!g || !o || which < 0 || which > 2) return fail(g, RT_ERR_INVALID_ARG, "rt_set_opacity: bad argument");
    OpacDev d;
    memset(&d, 0, sizeof(d));
    d.set = 1;
    d.kind = o->kind;
    if (o->kind == 0) {
        if (!(o->rho0 > 0.0) || !(o->T0 > 0.0) || !(o->kmax >= o->kmin) || !(o->kmin >= 0.0) || !(o->kappa0 >= 0.0))
            return fail(g, RT_ERR_INVALID_ARG, "rt_set_opacity: power law needs rho0, T0 > 0, kappa0 >= 0, 0 <= kmin <= kmax");
        d.kappa0 = o->kappa0;
        d.irho0 = 1.0 / o->rho0;
        d.iT0 = 1.0 / o->T0;
        d.a = o->a;
        d.b = o->b;
        d.kmin = o->kmin;
        d.kmax = o->kmax;
        d.n2a = half_int_exponent(o->a);
        d.n2b = half_int_exponent(o->b);
        d.fast = (d.n2a != INT_MIN && d.n2b != INT_MIN && abs(d.n2a) <= 15 && abs(d.n2b) <= 15) ? 1 : 0;
    } else if (o->kind == 1) {
        if (!o->log10_kappa || o->n_lT < 2 || o->n_lrho < 1)
            return fail(g, RT_ERR_INVALID_ARG, "rt_set_opacity: table needs n_lT >= 2, n_lrho >= 2 (or == 1) and data");
        if (!(o->lT_max > o->lT_min) || !(o->T_unit > 0.0)) return fail(g, RT_ERR_INVALID_ARG, "rt_set_opacity: bad T axis");
        if (o->n_lrho > 1 && (!(o->lrho_max > o->lrho_min) || !(o->rho_unit > 0.0)))
            return fail(g, RT_ERR_INVALID_ARG, "rt_set_opacity: bad rho axis");
        d.n_lrho = o->n_lrho;
        d.n_lT = o->n_lT;
        d.lrho_min = o->lrho_min;
        d.lrho_max = o->lrho_max;
        d.lT_min = o->lT_min;
        d.lT_max = o->lT_max;
        d.su = o->n_lrho > 1 ? (double)(o->n_lrho - 1) / (o->lrho_max - o->lrho_min) : 0.0;
        d.sv = (double)(o->n_lT - 1) / (o->lT_max - o->lT_min);
        d.rho_unit = o->rho_unit;
        d.T_unit = o->T_unit;
        const size_t cnt = (size_t)o->n_lT * (size_t)o->n_lrho;
        g->table_host[which].assign(o->log10_kappa, o->log10_kappa + cnt);
        RT_CUDA(g, cudaStreamSynchronize(g->stream));  // the old table may still be in use
        cudaFree(g->table_dev[which]);
        g->table_dev[which] = nullptr;
        RT_CUDA(g, cudaMalloc(&g->table_dev[which], cnt * sizeof(double)));
        RT_CUDA(g, cudaMemcpyAsync(g->table_dev[which], g->table_host[which].data(), cnt * sizeof(double),
                                   cudaMemcpyHostToDevice, g->stream));
        RT_CUDA(g, cudaStreamSynchronize(g->stream));
        d.tab = g->table_dev[which];
    } else {
        return fail(g, RT_ERR_INVALID_ARG, "rt_set_opacity: kind must be 0 (power law) or 1 (table)");
    }
    g->opac[which] = d;
    g->opac_host[which] = *o;
    g->opac_host[which].log10_kappa = nullptr;
    g->same_PR = same_law(g, RT_OPAC_PLANCK, RT_OPAC_ROSSELAND) ? 1 : 0;
    return RT_OK;
}

// which table opacities among `members` (RT_OPAC_* indices) can share log10(rho rho_unit), log10(T T_unit)
static OpacSet opac_set(const rt_grid* g, const int* members, int nm) {
    OpacSet os = {0, -1};
    int ntab = 0;
    for (int a = 0; a < nm; ++a) {
        const int w = members[a];
        if (!g->opac[w].set || g->opac[w].kind != 1) continue;
        ++ntab;
        if (os.src < 0) {
            os.src = w;
            continue;
        }
        const OpacDev &x = g->opac[os.src], &y = g->opac[w];
        if (x.T_unit != y.T_unit || (x.n_lrho > 1) != (y.n_lrho > 1) || (x.n_lrho > 1 && x.rho_unit != y.rho_unit)) return OpacSet{0, -1};
    }
    os.share = ntab >= 2 ? 1 : 0;
    return os;
}

// ------------------------------------------------------------------------------------------------
static int32_t launch_fill_ghosts(rt_grid* g, double* const U[4]) {
    const GridDev& D = g->dev;
    Fields4 F;
    for (int q = 0; q < 4; ++q) F.q[q] = U[q];
    for (int d = 0; d < 3; ++d) {
        if (D.gh[d] == 0) continue;
        if (D.bc[2 * d] == RT_BC_FIXED && D.bc[2 * d + 1] == RT_BC_FIXED) continue;
        long long tot = 4;
        for (int e = 0; e < 3; ++e)
            if (e != d) tot *= (e < d) ? D.nt[e] : D.n[e];
        const int nb = (int)((tot + 255) / 256 > 4096 ? 4096 : (tot + 255) / 256);
        {
            ProfScope ps(g, RT_K_GHOST);
            k_fill_ghosts<<<nb, 256, 0, g->stream>>>(D, F, d);
        }
        RT_LAUNCH_CHECK(g);
    }
    return RT_OK;
}

// blocks of 256 threads for the face-normal ghost fill (0: nothing to fill)
static int fill_faces_blocks(const GridDev& D) {
    long long tot = 0;
    for (int d = 0; d < 3; ++d) {
        if (D.gh[d] == 0 || (D.bc[2 * d] == RT_BC_FIXED && D.bc[2 * d + 1] == RT_BC_FIXED)) continue;
        long long c = 2;  // work items: (transverse cell, side), both layers each
        for (int e = 0; e < 3; ++e)
            if (e != d) c *= D.n[e];
        tot += c;
    }
    return (int)((tot + 255) / 256 > 8192 ? 8192 : (tot + 255) / 256);
}

// face-normal ghosts of all active axes in one launch (the sub-step kernels read nothing else)
static int32_t launch_fill_faces(rt_grid* g, double* const U[4], cudaStream_t st = nullptr) {
    if (!st) st = g->stream;
    const GridDev& D = g->dev;
    Fields4 F;
    for (int q = 0; q < 4; ++q) F.q[q] = U[q];
    const int nb = fill_faces_blocks(D);
    if (nb == 0) return RT_OK;
    {
        ProfScope ps(g, RT_K_GHOST, st);
        k_fill_faces<<<nb, 256, 0, st>>>(D, F);
    }
    RT_LAUNCH_CHECK(g);
    return RT_OK;
}

extern "C" int32_t rt_fill_ghosts(rt_grid* g, double* const U[4]) {
    DeviceGuard dg_(g);
    if (!g || !U) return fail(g, RT_ERR_INVALID_ARG, "rt_fill_ghosts: null argument");
    for (int q = 0; q < 4; ++q)
        if (!aligned8(U[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_fill_ghosts: U[%d] null or misaligned", q);
    return launch_fill_ghosts(g, U);
}

template <bool HLL, bool THICK, bool CURVI>
static void launch_x(rt_grid* g, const SweepArgs& a) {
    const GridDev& D = g->dev;
    const int nchunk = (D.n[0] + kXOut - 1) / kXOut;
    const long long ntask = (long long)nchunk * D.n[1] * D.n[2];
    const long long nblk = (ntask + 3) / 4;
    k_sweep_x<HLL, THICK, CURVI><<<(unsigned)nblk, 128, 0, g->stream>>>(D, a, nchunk, ntask);
}

template <int DIR, bool HLL, bool THICK, bool CURVI>
static void launch_march(rt_grid* g, const SweepArgs& a) {
    const GridDev& D = g->dev;
    constexpr int EO = (DIR == 1) ? 2 : 1;
    int bx = D.n[0] >= 128 ? 128 : ((D.n[0] + 31) / 32) * 32;
    int seg = g->march_len > 0 ? g->march_len : 32;
    if (seg > D.n[DIR]) seg = D.n[DIR];
    dim3 grid((D.n[0] + bx - 1) / bx, D.n[EO], (D.n[DIR] + seg - 1) / seg);
    k_sweep_march<DIR, HLL, THICK, CURVI><<<grid, bx, 0, g->stream>>>(D, a, seg);
}

template <bool HLL, bool THICK, bool CURVI>
static void launch_dir(rt_grid* g, int d, const SweepArgs& a) {
    if (d == 0) launch_x<HLL, THICK, CURVI>(g, a);
    else if (d == 1) launch_march<1, HLL, THICK, CURVI>(g, a);
    else launch_march<2, HLL, THICK, CURVI>(g, a);
}

static void launch_sweep(rt_grid* g, int d, bool hll, bool thick, bool curvi, const SweepArgs& a) {
    const int key = (hll ? 4 : 0) | (thick ? 2 : 0) | (curvi ? 1 : 0);
    switch (key) {
        case 0: launch_dir<false, false, false>(g, d, a); break;
        case 1: launch_dir<false, false, true>(g, d, a); break;
        case 2: launch_dir<false, true, false>(g, d, a); break;
        case 3: launch_dir<false, true, true>(g, d, a); break;
        case 4: launch_dir<true, false, false>(g, d, a); break;
        case 5: launch_dir<true, false, true>(g, d, a); break;
        case 6: launch_dir<true, true, false>(g, d, a); break;
        default: launch_dir<true, true, true>(g, d, a); break;
    }
}

// chi is ONE half-integer power law (kappa_R fast, no scattering) and kappa_P, when asked for, is the same law or another
// fast law with the same rho0, T0: the pre-pass takes its lean path (k_thick_limit<1>)
static bool lean_laws(const rt_grid* g, bool with_kp) {
    const OpacDev &oP = g->opac[RT_OPAC_PLANCK], &oR = g->opac[RT_OPAC_ROSSELAND], &oS = g->opac[RT_OPAC_SCATTER];
    bool lean = oR.set && oR.kind == 0 && oR.fast && !oS.set;
    if (with_kp && !g->same_PR) lean = lean && oP.set && oP.kind == 0 && oP.fast && oP.irho0 == oR.irho0 && oP.iT0 == oR.iT0;
    return lean;
}

// with_kp: also write rho kappa_P per cell into g->kpr (fused sub-step: the implicit half then evaluates no opacity)
// Ufill: also fill the face-normal ghosts of these four fields, in the same launch (k_thick_limit_faces)
static int32_t launch_thick_limit(rt_grid* g, const double* rho, const double* T, bool with_kp = false,
                                  double* const* Ufill = nullptr) {
    const GridDev& D = g->dev;
    // ghosts the kernel never writes (beyond the first face-normal layer) are never used either: zero them once
    if (!g->lim) {
        RT_CUDA(g, cudaMalloc(&g->lim, (size_t)D.ntot * sizeof(double)));
        RT_CUDA(g, cudaMemsetAsync(g->lim, 0, (size_t)D.ntot * sizeof(double), g->stream));
    }
    if (with_kp && !g->kpr) {
        RT_CUDA(g, cudaMalloc(&g->kpr, (size_t)D.ntot * sizeof(double)));
        RT_CUDA(g, cudaMemsetAsync(g->kpr, 0, (size_t)D.ntot * sizeof(double), g->stream));
    }
    // block width (<= 256, a multiple of 32) that wastes the fewest lanes on a row of n1 cells
    int bx = 256;
    {
        long long best = -1;
        for (int cand = 256; cand >= 64; cand -= 32) {
            const long long lanes = (long long)((D.n[0] + cand - 1) / cand) * cand;
            if (best < 0 || lanes < best) {
                best = lanes;
                bx = cand;
            }
        }
    }
    // x2 rows per block: kThickRows, or (lean power laws: register batches of kThickRows rows, the next batch prefetched
    // into L2) four times as many where that still leaves >= 16 blocks per SM
    int rpb = kThickRows;
    if (lean_laws(g, with_kp)) {
        rpb = 4 * kThickRows;
        while (rpb > kThickRows && (long long)((D.n[0] + bx - 1) / bx) * ((D.n[1] + rpb - 1) / rpb) * D.n[2] < 16LL * 148) rpb /= 2;
    }
    dim3 grid((D.n[0] + bx - 1) / bx, (D.n[1] + rpb - 1) / rpb, D.n[2]);
    int nbg = Ufill ? fill_faces_blocks(D) : 0;
    const long long nthick = (long long)grid.x * grid.y * grid.z;
    if (nbg > 0 && nthick + nbg >= (1LL << 31)) {  // too many blocks for one 1-D grid: two launches
        const int32_t rcf = launch_fill_faces(g, Ufill);
        if (rcf != RT_OK) return rcf;
        nbg = 0;
    }
    {
        ProfScope ps(g, RT_K_THICK);
        const OpacDev &oP = g->opac[RT_OPAC_PLANCK], &oR = g->opac[RT_OPAC_ROSSELAND], &oS = g->opac[RT_OPAC_SCATTER];
        const int m2[2] = {RT_OPAC_ROSSELAND, RT_OPAC_SCATTER};
        const int m3[3] = {RT_OPAC_PLANCK, RT_OPAC_ROSSELAND, RT_OPAC_SCATTER};
        const OpacSet os = with_kp ? opac_set(g, m3, 3) : opac_set(g, m2, 2);
        const bool lean = lean_laws(g, with_kp);
        const bool second = with_kp && !g->same_PR;
        double* kpr = with_kp ? g->kpr : nullptr;
        LeanLaws L;
        memset(&L, 0, sizeof(L));
        if (lean) {
            L.irho0 = oR.irho0;
            L.iT0 = oR.iT0;
            L.two = second ? 1 : 0;
            L.k0[0] = oR.kappa0; L.kmin[0] = oR.kmin; L.kmax[0] = oR.kmax; L.na[0] = oR.n2a; L.nb[0] = oR.n2b;
            if (second) {
                L.k0[1] = oP.kappa0; L.kmin[1] = oP.kmin; L.kmax[1] = oP.kmax; L.na[1] = oP.n2a; L.nb[1] = oP.n2b;
                L.same_ab = (oP.n2a == oR.n2a && oP.n2b == oR.n2b) ? 1 : 0;
            }
        }
        // two 2-D tables on the same axes and units (or one), no scattering: the table-pair path
        TablePair tp;
        memset(&tp, 0, sizeof(tp));
        bool pair = !lean && oR.set && oR.kind == 1 && oR.n_lrho > 1 && !oS.set;
        if (pair && second)
            pair = oP.set && oP.kind == 1 && oP.n_lrho == oR.n_lrho && oP.n_lT == oR.n_lT && oP.lrho_min == oR.lrho_min &&
                   oP.lrho_max == oR.lrho_max && oP.lT_min == oR.lT_min && oP.lT_max == oR.lT_max && oP.rho_unit == oR.rho_unit &&
                   oP.T_unit == oR.T_unit;
        if (pair) {
            tp.tabR = oR.tab;
            tp.tabP = second ? oP.tab : nullptr;
            tp.n_lrho = oR.n_lrho; tp.n_lT = oR.n_lT;
            tp.lrho_min = oR.lrho_min; tp.lrho_max = oR.lrho_max; tp.lT_min = oR.lT_min; tp.lT_max = oR.lT_max;
            tp.su = oR.su; tp.sv = oR.sv; tp.rho_unit = oR.rho_unit; tp.T_unit = oR.T_unit;
        }
        if (nbg > 0) {
            // the ghost fill rides in the same launch (its blocks are sized for 256 threads; bx <= 256 of them only makes
            // their grid-stride loops a little longer)
            Fields4 F;
            for (int q = 0; q < 4; ++q) F.q[q] = Ufill[q];
            const unsigned nblk = (unsigned)(nthick + nbg);
            const int gx = (int)grid.x, gy = (int)grid.y;
            if (lean && rpb > kThickRows)
                k_thick_limit_faces<3><<<nblk, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, F, nbg, gx, gy, rpb);
            else if (lean)
                k_thick_limit_faces<1><<<nblk, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, F, nbg, gx, gy, rpb);
            else if (pair)
                k_thick_limit_faces<2><<<nblk, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, F, nbg, gx, gy, rpb);
            else
                k_thick_limit_faces<0><<<nblk, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, F, nbg, gx, gy, rpb);
        } else {
            if (lean && rpb > kThickRows)
                k_thick_limit<3><<<grid, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, rpb);
            else if (lean)
                k_thick_limit<1><<<grid, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, rpb);
            else if (pair)
                k_thick_limit<2><<<grid, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, rpb);
            else
                k_thick_limit<0><<<grid, bx, 0, g->stream>>>(D, oR, oS, os, rho, T, g->lim, oP, g->same_PR, kpr, L, tp, rpb);
        }
    }
    RT_LAUNCH_CHECK(g);
    return RT_OK;
}

// explicit half; the time step is dt (host) or, when dt_dev != nullptr, the device double *dt_dev
static int32_t explicit_impl(rt_grid* g, double dt, const double* dt_dev, const double* rho, const double* T,
                             double* const U_in[4], double* const U_out[4]) {
    if (g) ProfScope::trim(g);
    if (!g || !U_in || !U_out) return fail(g, RT_ERR_INVALID_ARG, "rt_explicit_step: null argument");
    if (!g->have_par) return fail(g, RT_ERR_BAD_STATE, "rt_explicit_step: rt_set_params has not been called");
    if (!dt_dev && (!(dt > 0.0) || !isfinite(dt))) return fail(g, RT_ERR_INVALID_ARG, "rt_explicit_step: dt must be finite and > 0");
    for (int q = 0; q < 4; ++q)
        if (!aligned8(U_in[q]) || !aligned8(U_out[q]) || U_in[q] == U_out[q])
            return fail(g, RT_ERR_INVALID_ARG, "rt_explicit_step: U_in/U_out[%d] null, misaligned or aliased", q);
    const bool thick = g->par.thick_limit != 0;
    if (thick && (!aligned8(rho) || !aligned8(T))) return fail(g, RT_ERR_INVALID_ARG, "rt_explicit_step: thick_limit needs rho and T");
    const GridDev& D = g->dev;

    int32_t rc = launch_fill_ghosts(g, U_in);
    if (rc != RT_OK) return rc;

    if (thick) {
        rc = launch_thick_limit(g, rho, T);
        if (rc != RT_OK) return rc;
    }

    SweepArgs a;
    for (int q = 0; q < 4; ++q) {
        a.uin[q] = U_in[q];
        a.uout[q] = U_out[q];
    }
    a.lim = thick ? g->lim : nullptr;
    a.dtc = dt * g->par.chat;
    a.dt_dev = dt_dev;
    a.chat = g->par.chat;
    a.rusanov = g->par.solver == RT_SOLVER_RUSANOV;
    a.fix = g->face_fix;
    a.recon = g->recon;
    a.limo3_r = g->limo3_r;
    const bool hll = g->par.solver != RT_SOLVER_GLF;  // HLL and Rusanov need the wave speeds
    const bool curvi = D.geometry != RT_CARTESIAN;
    if (D.gh[0] == 0) {
        // no x1 sweep: start the accumulation from a copy of U^n (rare: grids with n1 == 1)
        for (int q = 0; q < 4; ++q)
            RT_CUDA(g, cudaMemcpyAsync(U_out[q], U_in[q], (size_t)D.ntot * sizeof(double), cudaMemcpyDeviceToDevice, g->stream));
    }
    for (int d = 0; d < 3; ++d) {
        if (D.gh[d] == 0) continue;
        {
            ProfScope ps(g, RT_K_SWEEP1 + d);
            launch_sweep(g, d, hll, thick, curvi, a);
        }
        RT_LAUNCH_CHECK(g);
    }
    return RT_OK;
}

extern "C" int32_t rt_explicit_step(rt_grid* g, double dt, const double* rho, const double* T, double* const U_in[4],
                                    double* const U_out[4]) {
    DeviceGuard dg_(g);
    return explicit_impl(g, dt, nullptr, rho, T, U_in, U_out);
}

// implicit half; with_cfl: fold the step-10 rate of the updated state into the scratch word and finalise
// dt_next_dev = cfl / max rate with a one-thread kernel
static int32_t implicit_impl(rt_grid* g, double dt, const double* dt_dev, const double* rho, double* T, double* const mom[3],
                             double* const U[4], bool with_cfl, double cfl, double* dt_next_dev) {
    if (!g || !U || !aligned8(rho) || !aligned8(T)) return fail(g, RT_ERR_INVALID_ARG, "rt_implicit_step: null or misaligned argument");
    if (!g->have_par) return fail(g, RT_ERR_BAD_STATE, "rt_implicit_step: rt_set_params has not been called");
    if (!dt_dev && (!(dt > 0.0) || !isfinite(dt))) return fail(g, RT_ERR_INVALID_ARG, "rt_implicit_step: dt must be finite and > 0");
    if (with_cfl && (!aligned8(dt_next_dev) || !(cfl > 0.0) || !isfinite(cfl)))
        return fail(g, RT_ERR_INVALID_ARG, "rt_implicit_step_cfl: cfl must be finite and > 0 and dt_next_device non-null");
    for (int q = 0; q < 4; ++q)
        if (!aligned8(U[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_implicit_step: U[%d] null or misaligned", q);
    const bool feedback = g->par.feedback_momentum && mom != nullptr;
    if (feedback)
        for (int q = 0; q < 3; ++q)
            if (!aligned8(mom[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_implicit_step: mom[%d] null or misaligned", q);
    const GridDev& D = g->dev;
    ImplicitArgs a;
    for (int q = 0; q < 4; ++q) a.U[q] = U[q];
    a.rho = rho;
    a.T = T;
    for (int q = 0; q < 3; ++q) a.mom[q] = feedback ? mom[q] : nullptr;
    a.dt = dt;
    a.dt_dev = dt_dev;
    a.scr = g->scr;
    a.feedback = feedback;
    a.same_PR = g->same_PR;
    {
        const int members[3] = {RT_OPAC_PLANCK, RT_OPAC_ROSSELAND, RT_OPAC_SCATTER};
        a.os = opac_set(g, members, 3);
    }
    a.ichat = 1.0 / g->par.chat;
    a.counters = g->counters;
    a.divfirr = g->divfirr;
    for (int q = 0; q < 4; ++q) a.avgU[q] = nullptr;
    a.avgT = nullptr;
    for (int q = 0; q < 3; ++q) a.avgm[q] = nullptr;
    a.Tout = a.T;
    for (int q = 0; q < 3; ++q) a.mout[q] = a.mom[q];
    ParamsDev P = {g->par.chat, g->par.c, g->par.a_R, g->par.c_v, g->par.E_floor, g->par.solver, g->par.thick_limit,
                   g->par.feedback_momentum};
    const int bx = D.n[0] >= 128 ? 128 : ((D.n[0] + 31) / 32) * 32;
    dim3 grid((D.n[0] + bx - 1) / bx, D.n[1], D.n[2]);
    {
        ProfScope ps(g, RT_K_IMPLICIT);
        if (feedback && with_cfl)
            k_implicit<true, true><<<grid, bx, 0, g->stream>>>(D, P, g->opac[0], g->opac[1], g->opac[2], a);
        else if (feedback)
            k_implicit<true, false><<<grid, bx, 0, g->stream>>>(D, P, g->opac[0], g->opac[1], g->opac[2], a);
        else if (with_cfl)
            k_implicit<false, true><<<grid, bx, 0, g->stream>>>(D, P, g->opac[0], g->opac[1], g->opac[2], a);
        else
            k_implicit<false, false><<<grid, bx, 0, g->stream>>>(D, P, g->opac[0], g->opac[1], g->opac[2], a);
    }
    RT_LAUNCH_CHECK(g);
    if (with_cfl) {
        {
            ProfScope ps(g, RT_K_CFL);
            k_cfl_finalize<<<1, 1, 0, g->stream>>>(g->scr, cfl, dt_next_dev);
        }
        RT_LAUNCH_CHECK(g);
    }
    return RT_OK;
}

extern "C" int32_t rt_set_reconstruction(rt_grid* g, int32_t kind, double r) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    if ((kind != RT_RECON_PLM && kind != RT_RECON_LIMO3) || !isfinite(r))
        return fail(g, RT_ERR_INVALID_ARG, "rt_set_reconstruction: unknown kind %d or non-finite r", kind);
    g->recon = kind;
    g->limo3_r = r;
    return RT_OK;
}

extern "C" int32_t rt_set_face_fix(rt_grid* g, int32_t mode) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    if (mode < RT_FIX_FPRESERVING || mode > RT_FIX_CLIP) return fail(g, RT_ERR_INVALID_ARG, "rt_set_face_fix: unknown mode %d", mode);
    g->face_fix = mode;
    return RT_OK;
}

extern "C" int32_t rt_irradiation_radial(rt_grid* g, double L0, double kappa_irr, double tau_in, const double* rho,
                                         double* tau_hi, double* div_firr) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    if (!aligned8(rho) || !aligned8(div_firr) || (tau_hi && !aligned8(tau_hi)))
        return fail(g, RT_ERR_INVALID_ARG, "rt_irradiation_radial: null or misaligned pointer");
    if (g->dev.geometry == RT_CYLINDRICAL) return fail(g, RT_ERR_INVALID_ARG, "rt_irradiation_radial: x1 rays need a spherical or Cartesian grid");
    if (!isfinite(L0) || !isfinite(kappa_irr) || !isfinite(tau_in) || !(kappa_irr >= 0.0) || !(tau_in >= 0.0))
        return fail(g, RT_ERR_INVALID_ARG, "rt_irradiation_radial: L0 finite, kappa_irr >= 0 and tau_in >= 0 required");
    const long long rays = (long long)g->dev.n[1] * g->dev.n[2];
    k_irradiation_radial<<<(unsigned)((rays + 3) / 4), 128, 0, g->stream>>>(g->dev, L0, kappa_irr, tau_in, rho, tau_hi, div_firr);
    RT_LAUNCH_CHECK(g);
    return RT_OK;
}

extern "C" int32_t rt_set_irradiation(rt_grid* g, const double* div_firr) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    if (div_firr && !aligned8(div_firr)) return fail(g, RT_ERR_INVALID_ARG, "rt_set_irradiation: misaligned pointer");
    g->divfirr = div_firr;
    return RT_OK;
}

extern "C" int32_t rt_implicit_step(rt_grid* g, double dt, const double* rho, double* T, double* const mom[3], double* const U[4]) {
    DeviceGuard dg_(g);
    return implicit_impl(g, dt, nullptr, rho, T, mom, U, false, 0.0, nullptr);
}

extern "C" int32_t rt_implicit_step_cfl(rt_grid* g, double dt, const double* rho, double* T, double* const mom[3],
                                        double* const U[4], double cfl, double* dt_next_device) {
    DeviceGuard dg_(g);
    return implicit_impl(g, dt, nullptr, rho, T, mom, U, true, cfl, dt_next_device);
}

// ------------------------------------------------------------------------------------------------
// Fused sub-step (3-D grids): ghost fill -> thick-limit pre-pass -> k_substep_fused -> k_cfl_finalize
// cuTensorMapEncodeTiled through the runtime's driver entry point lookup: no link-time dependency on libcuda
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        cudaGetLastError();
    }
    return fn;
}

// TMA descriptors of the staged arrays: ghosted (nt1, nt2, nt3) fp64 tensors, box 34 x FPH x 1, zero fill outside.
// false when the TMA cannot address them (row pitch or base not a multiple of 16 B, or no encoder).
static bool fused_make_maps(const rt_grid* g, const FusedArgs& a, int narr, FusedMaps* maps) {
    const GridDev& D = g->dev;
    if ((D.nt[0] & 1) != 0) return false;
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const cuuint64_t gdim[3] = {(cuuint64_t)D.nt[0], (cuuint64_t)D.nt[1], (cuuint64_t)D.nt[2]};
    const cuuint64_t gstr[2] = {(cuuint64_t)D.nt[0] * 8u, (cuuint64_t)D.nt[0] * (cuuint64_t)D.nt[1] * 8u};
    const cuuint32_t box[3] = {(cuuint32_t)FPW, (cuuint32_t)FPH, 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    for (int q = 0; q < narr; ++q) {
        if ((reinterpret_cast<uintptr_t>(a.src[q]) & 15u) != 0) return false;
        if (enc(&maps->m[q], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(a.src[q]), gdim, gstr, box, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    return true;
}

template <bool HLL, bool THICK, bool CURVI, bool FEEDBACK, bool RUS, bool HASZ, int VMODE>
static cudaError_t launch_fused_z(rt_grid* g, const ParamsDev& P, const FusedArgs& a, const FusedMaps& maps, dim3 grid, int seglen) {
    auto kern = k_substep_fused<HLL, THICK, CURVI, FEEDBACK, RUS, HASZ, VMODE>;
    // the attribute is per device (and per instantiation: this function is a template)
    static bool attr_done[64] = {false};
    const int dev = g->device >= 0 && g->device < 64 ? g->device : 0;
    if (!attr_done[dev] || g->device >= 64) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmemBytes);
        if (e != cudaSuccess) return e;
        attr_done[dev] = true;
    }
    kern<<<grid, dim3(32, FNY), kFusedSmemBytes, g->stream>>>(g->dev, P, g->opac[0], g->opac[1], g->opac[2], a, maps, seglen);
    return cudaSuccess;
}

// x3 active (3-D) or not (2-D); the comparison face fixes (a.fix != 0; never with the Rusanov solver: fused_eligible)
template <bool HLL, bool THICK, bool CURVI, bool FEEDBACK, bool RUS = false>
static cudaError_t launch_fused_t(rt_grid* g, const ParamsDev& P, const FusedArgs& a, const FusedMaps& maps, dim3 grid, int seglen) {
    // VMODE (rt_kernels_fused.cuh): 2 = run-time face fix (+ RK2 options), 1 = RK2 average, 0 = neither
    if (!RUS && a.fix != 0)
        return g->dev.gh[2] > 0 ? launch_fused_z<HLL, THICK, CURVI, FEEDBACK, false, true, 2>(g, P, a, maps, grid, seglen)
                                : launch_fused_z<HLL, THICK, CURVI, FEEDBACK, false, false, 2>(g, P, a, maps, grid, seglen);
    if (!RUS && a.im.avgU[0] != nullptr)
        return g->dev.gh[2] > 0 ? launch_fused_z<HLL, THICK, CURVI, FEEDBACK, false, true, 1>(g, P, a, maps, grid, seglen)
                                : launch_fused_z<HLL, THICK, CURVI, FEEDBACK, false, false, 1>(g, P, a, maps, grid, seglen);
    return g->dev.gh[2] > 0 ? launch_fused_z<HLL, THICK, CURVI, FEEDBACK, RUS, true, 0>(g, P, a, maps, grid, seglen)
                            : launch_fused_z<HLL, THICK, CURVI, FEEDBACK, RUS, false, 0>(g, P, a, maps, grid, seglen);
}

static cudaError_t launch_fused(rt_grid* g, bool hll, bool thick, bool curvi, bool feedback, const ParamsDev& P,
                                const FusedArgs& a, const FusedMaps& maps, dim3 grid, int seglen) {
    const int key = (hll ? 8 : 0) | (thick ? 4 : 0) | (curvi ? 2 : 0) | (feedback ? 1 : 0);
    if (g->par.solver == RT_SOLVER_RUSANOV) {
        switch (key & 7) {
#define RT_FUSED_CASE(K, B, C_, D_) case K: return launch_fused_t<true, B, C_, D_, true>(g, P, a, maps, grid, seglen);
            RT_FUSED_CASE(0, false, false, false)
            RT_FUSED_CASE(1, false, false, true)
            RT_FUSED_CASE(2, false, true, false)
            RT_FUSED_CASE(3, false, true, true)
            RT_FUSED_CASE(4, true, false, false)
            RT_FUSED_CASE(5, true, false, true)
            RT_FUSED_CASE(6, true, true, false)
            default: return launch_fused_t<true, true, true, true, true>(g, P, a, maps, grid, seglen);
#undef RT_FUSED_CASE
        }
    }
    switch (key) {
#define RT_FUSED_CASE(K, A, B, C_, D_) case K: return launch_fused_t<A, B, C_, D_>(g, P, a, maps, grid, seglen);
        RT_FUSED_CASE(0, false, false, false, false)
        RT_FUSED_CASE(1, false, false, false, true)
        RT_FUSED_CASE(2, false, false, true, false)
        RT_FUSED_CASE(3, false, false, true, true)
        RT_FUSED_CASE(4, false, true, false, false)
        RT_FUSED_CASE(5, false, true, false, true)
        RT_FUSED_CASE(6, false, true, true, false)
        RT_FUSED_CASE(7, false, true, true, true)
        RT_FUSED_CASE(8, true, false, false, false)
        RT_FUSED_CASE(9, true, false, false, true)
        RT_FUSED_CASE(10, true, false, true, false)
        RT_FUSED_CASE(11, true, false, true, true)
        RT_FUSED_CASE(12, true, true, false, false)
        RT_FUSED_CASE(13, true, true, false, true)
        RT_FUSED_CASE(14, true, true, true, false)
        default: return launch_fused_t<true, true, true, true>(g, P, a, maps, grid, seglen);
#undef RT_FUSED_CASE
    }
}

// x3 segment length of the fused kernel: the CTA count should fill whole waves of 2 CTAs per SM, with segments
// long enough that the two half-work planes at the segment ends stay a small share.
static int fused_segment_length(const rt_grid* g, int tiles) {
    const int n3 = g->dev.n[2];
    if (g->fused_seg > 0) return g->fused_seg < n3 ? g->fused_seg : n3;
    int dev = 0, nsm = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const double slots = 2.0 * nsm;
    // measured on B200 (C4): segments of 32-43 planes beat 64-128 by ~2.5 % (finer tail), shorter ones pay the two
    // half-work planes at the segment ends; among lengths 12..48 take the best wave fill x end overhead
    if (n3 <= 12) return n3;
    int best = n3 < 32 ? n3 : 32;
    double best_score = -1.0;
    // 12..48: small grids (C3: 80 tiles) need short segments to fill the machine, large ones are flat in this range
    for (int len = 12; len <= 48 && len <= n3; ++len) {
        const int ns = (n3 + len - 1) / len;
        const double ctas = (double)tiles * ns;
        const double fill = ctas / (ceil(ctas / slots) * slots);                 // tail effect
        const double work = (double)n3 / ((double)n3 + 0.7 * ns);                // segment-end overhead
        const double ragged = (double)n3 / ((double)ns * len);                   // last segment shorter than the others
        const double score = fill * work * (0.5 + 0.5 * ragged);
        if (score > best_score) {
            best_score = score;
            best = len;
        }
    }
    return best;
}

static bool fused_eligible(const rt_grid* g) {
    const GridDev& D = g->dev;
    // the comparison face fixes (rt_set_face_fix) run in the fused kernel too, except with the Rusanov solver
    // LimO3 (rt_set_reconstruction) exists in the per-direction kernels and the 1-D kernel only
    return g->fused_seg >= 0 && g->recon == RT_RECON_PLM &&
           (g->face_fix == RT_FIX_FPRESERVING || g->par.solver != RT_SOLVER_RUSANOV) && D.gh[0] > 0 &&
           D.gh[1] > 0 && D.ntot < (1LL << 31);  // 32-bit element offsets inside the kernel
}

// RK2: what the second stage averages its result with (fused into its stores), and where the new time step goes
struct RkAvg {
    const double* U[4];   // average the result with these (nullptr: no average: first stage)
    const double* T;
    const double* m[3];
    double* Tout;         // updated T, m go here instead of in place (nullptr: in place)
    double* mout[3];
    double* dt_out;       // the new time step (nullptr: dt_device)
};

static int32_t fused_impl(rt_grid* g, double* dt_device, double cfl, const double* rho, double* T, double* const mom[3],
                          double* const U_in[4], double* const U_out[4], const RkAvg* avg = nullptr) {
    ProfScope::trim(g);
    if (!U_in || !U_out) return fail(g, RT_ERR_INVALID_ARG, "rt_substep: null argument");
    if (!g->have_par) return fail(g, RT_ERR_BAD_STATE, "rt_substep: rt_set_params has not been called");
    for (int q = 0; q < 4; ++q)
        if (!aligned8(U_in[q]) || !aligned8(U_out[q]) || U_in[q] == U_out[q])
            return fail(g, RT_ERR_INVALID_ARG, "rt_substep: U_in/U_out[%d] null, misaligned or aliased", q);
    const bool feedback = g->par.feedback_momentum && mom != nullptr;
    if (feedback)
        for (int q = 0; q < 3; ++q)
            if (!aligned8(mom[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_substep: mom[%d] null or misaligned", q);
    const GridDev& D = g->dev;
    const bool thick = g->par.thick_limit != 0;

    // the ghost fill and, with the thick limit, the pre-pass: one launch (k_thick_limit_faces)
    int32_t rc = thick ? launch_thick_limit(g, rho, T, true, U_in) : launch_fill_faces(g, U_in);
    if (rc != RT_OK) return rc;
    FusedArgs a;
    for (int q = 0; q < 4; ++q) {
        a.src[q] = U_in[q];
        a.im.U[q] = U_out[q];
    }
    a.src[4] = thick ? g->lim : nullptr;
    a.kpr = thick ? g->kpr : nullptr;
    a.chat = g->par.chat;
    a.fix = g->face_fix;
    a.im.rho = rho;
    a.im.T = T;
    for (int q = 0; q < 3; ++q) a.im.mom[q] = feedback ? mom[q] : nullptr;
    a.im.dt = 0.0;
    a.im.dt_dev = dt_device;
    a.im.scr = g->scr;
    a.im.feedback = feedback;
    a.im.same_PR = g->same_PR;
    {
        const int members[3] = {RT_OPAC_PLANCK, RT_OPAC_ROSSELAND, RT_OPAC_SCATTER};
        a.im.os = opac_set(g, members, 3);
    }
    a.im.ichat = 1.0 / g->par.chat;
    a.im.counters = g->counters;
    a.im.divfirr = g->divfirr;
    for (int q = 0; q < 4; ++q) a.im.avgU[q] = avg ? avg->U[q] : nullptr;
    a.im.avgT = avg ? avg->T : nullptr;
    for (int q = 0; q < 3; ++q) a.im.avgm[q] = (avg && feedback) ? avg->m[q] : nullptr;
    a.im.Tout = (avg && avg->Tout) ? avg->Tout : T;
    for (int q = 0; q < 3; ++q) a.im.mout[q] = feedback ? ((avg && avg->mout[q]) ? avg->mout[q] : mom[q]) : nullptr;
    ParamsDev P = {g->par.chat, g->par.c, g->par.a_R, g->par.c_v, g->par.E_floor, g->par.solver, g->par.thick_limit,
                   g->par.feedback_momentum};
    const int tx = (D.n[0] + FTX - 1) / FTX, ty = (D.n[1] + FTY - 1) / FTY;
    const int seglen = fused_segment_length(g, tx * ty);
    dim3 grid(tx, ty, (D.n[2] + seglen - 1) / seglen);
    FusedMaps maps;
    memset(&maps, 0, sizeof(maps));
    a.use_tma = 0;
    if (g->fused_tma_off == 0) {
        const int narr = thick ? 5 : 4;
        const rt_grid::MapEntry* hit = nullptr;
        for (const auto& e : g->map_cache) {
            bool same = e.narr == narr;
            for (int q = 0; q < narr && same; ++q) same = e.key[q] == a.src[q];
            if (same) {
                hit = &e;
                break;
            }
        }
        if (hit) {
            maps = hit->maps;
            a.use_tma = 1;
        } else if (fused_make_maps(g, a, narr, &maps)) {
            a.use_tma = 1;
            if (g->map_cache.size() >= 8) g->map_cache.erase(g->map_cache.begin());
            rt_grid::MapEntry e;
            memset(&e, 0, sizeof(e));
            for (int q = 0; q < narr; ++q) e.key[q] = a.src[q];
            e.narr = narr;
            e.maps = maps;
            g->map_cache.push_back(e);
        }
    }
    {
        ProfScope ps(g, RT_K_FUSED);
        cudaError_t e = launch_fused(g, g->par.solver != RT_SOLVER_GLF, thick, D.geometry != RT_CARTESIAN, feedback, P, a, maps, grid, seglen);
        if (e != cudaSuccess) return fail(g, RT_ERR_CUDA, "k_substep_fused attribute: %s", cudaGetErrorString(e));
    }
    RT_LAUNCH_CHECK(g);
    {
        ProfScope ps(g, RT_K_CFL);
        k_cfl_finalize<<<1, 1, 0, g->stream>>>(g->scr, cfl, (avg && avg->dt_out) ? avg->dt_out : dt_device);
    }
    RT_LAUNCH_CHECK(g);
    return RT_OK;
}

// Small 1-D grids: the whole sub-step in one launch of one CTA (k_substep_1d)
static bool oned_eligible(const rt_grid* g) {
    const GridDev& D = g->dev;
    return g->fused_seg >= 0 && D.gh[0] > 0 && D.gh[1] == 0 && D.gh[2] == 0 && D.n[0] >= 2 && D.n[0] <= K1D_MAXN;
}

template <bool HLL, bool THICK, bool CURVI>
static void launch_1d(rt_grid* g, bool feedback, const ParamsDev& P, const SweepArgs& sw, const ImplicitArgs& im, double cfl,
                      double* dt_out) {
    if (feedback)
        k_substep_1d<HLL, THICK, CURVI, true><<<1, K1D_NT, 0, g->stream>>>(g->dev, P, g->opac[0], g->opac[1], g->opac[2], sw, im, cfl, dt_out);
    else
        k_substep_1d<HLL, THICK, CURVI, false><<<1, K1D_NT, 0, g->stream>>>(g->dev, P, g->opac[0], g->opac[1], g->opac[2], sw, im, cfl, dt_out);
}

static int32_t oned_impl(rt_grid* g, double* dt_device, double cfl, const double* rho, double* T, double* const mom[3],
                         double* const U_in[4], double* const U_out[4]) {
    if (!U_in || !U_out) return fail(g, RT_ERR_INVALID_ARG, "rt_substep: null argument");
    if (!g->have_par) return fail(g, RT_ERR_BAD_STATE, "rt_substep: rt_set_params has not been called");
    for (int q = 0; q < 4; ++q)
        if (!aligned8(U_in[q]) || !aligned8(U_out[q]) || U_in[q] == U_out[q])
            return fail(g, RT_ERR_INVALID_ARG, "rt_substep: U_in/U_out[%d] null, misaligned or aliased", q);
    const bool feedback = g->par.feedback_momentum && mom != nullptr;
    if (feedback)
        for (int q = 0; q < 3; ++q)
            if (!aligned8(mom[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_substep: mom[%d] null or misaligned", q);
    const GridDev& D = g->dev;
    SweepArgs sw;
    for (int q = 0; q < 4; ++q) {
        sw.uin[q] = U_in[q];
        sw.uout[q] = U_out[q];
    }
    sw.lim = nullptr;
    sw.dtc = 0.0;
    sw.dt_dev = dt_device;
    sw.chat = g->par.chat;
    sw.rusanov = g->par.solver == RT_SOLVER_RUSANOV;
    sw.fix = g->face_fix;
    sw.recon = g->recon;
    sw.limo3_r = g->limo3_r;
    ImplicitArgs a;
    for (int q = 0; q < 4; ++q) a.U[q] = U_out[q];
    a.rho = rho;
    a.T = T;
    for (int q = 0; q < 3; ++q) a.mom[q] = feedback ? mom[q] : nullptr;
    a.dt = 0.0;
    a.dt_dev = dt_device;
    a.scr = g->scr;
    a.feedback = feedback;
    a.same_PR = g->same_PR;
    {
        const int members[3] = {RT_OPAC_PLANCK, RT_OPAC_ROSSELAND, RT_OPAC_SCATTER};
        a.os = opac_set(g, members, 3);
    }
    a.ichat = 1.0 / g->par.chat;
    a.counters = g->counters;
    a.divfirr = g->divfirr;
    for (int q = 0; q < 4; ++q) a.avgU[q] = nullptr;
    a.avgT = nullptr;
    for (int q = 0; q < 3; ++q) a.avgm[q] = nullptr;
    a.Tout = a.T;
    for (int q = 0; q < 3; ++q) a.mout[q] = a.mom[q];
    ParamsDev P = {g->par.chat, g->par.c, g->par.a_R, g->par.c_v, g->par.E_floor, g->par.solver, g->par.thick_limit,
                   g->par.feedback_momentum};
    const bool hll = g->par.solver != RT_SOLVER_GLF, thick = g->par.thick_limit != 0, curvi = D.geometry != RT_CARTESIAN;
    {
        ProfScope ps(g, RT_K_FUSED);
        const int key = (hll ? 4 : 0) | (thick ? 2 : 0) | (curvi ? 1 : 0);
        switch (key) {
            case 0: launch_1d<false, false, false>(g, feedback, P, sw, a, cfl, dt_device); break;
            case 1: launch_1d<false, false, true>(g, feedback, P, sw, a, cfl, dt_device); break;
            case 2: launch_1d<false, true, false>(g, feedback, P, sw, a, cfl, dt_device); break;
            case 3: launch_1d<false, true, true>(g, feedback, P, sw, a, cfl, dt_device); break;
            case 4: launch_1d<true, false, false>(g, feedback, P, sw, a, cfl, dt_device); break;
            case 5: launch_1d<true, false, true>(g, feedback, P, sw, a, cfl, dt_device); break;
            case 6: launch_1d<true, true, false>(g, feedback, P, sw, a, cfl, dt_device); break;
            default: launch_1d<true, true, true>(g, feedback, P, sw, a, cfl, dt_device); break;
        }
    }
    RT_LAUNCH_CHECK(g);
    return RT_OK;
}

extern "C" int32_t rt_substep(rt_grid* g, double* dt_device, double cfl, const double* rho, double* T, double* const mom[3],
                              double* const U_in[4], double* const U_out[4]) {
    DeviceGuard dg_(g);
    if (!g || !aligned8(dt_device)) return fail(g, RT_ERR_INVALID_ARG, "rt_substep: null or misaligned dt_device");
    if (!(cfl > 0.0) || !isfinite(cfl)) return fail(g, RT_ERR_INVALID_ARG, "rt_substep: cfl must be finite and > 0");
    if (!aligned8(rho) || !aligned8(T)) return fail(g, RT_ERR_INVALID_ARG, "rt_substep: rho / T null or misaligned");
    if (fused_eligible(g)) return fused_impl(g, dt_device, cfl, rho, T, mom, U_in, U_out);
    if (oned_eligible(g)) return oned_impl(g, dt_device, cfl, rho, T, mom, U_in, U_out);
    int32_t rc = explicit_impl(g, 0.0, dt_device, rho, T, U_in, U_out);
    if (rc != RT_OK) return rc;
    return implicit_impl(g, 0.0, dt_device, rho, T, mom, U_out, true, cfl, dt_device);
}

// internal form of rt_substep (arguments already validated by the callers' first use)
static int32_t substep_impl(rt_grid* g, double* dt_device, double cfl, const double* rho, double* T, double* const mom[3],
                            double* const U_in[4], double* const U_out[4]) {
    if (fused_eligible(g)) return fused_impl(g, dt_device, cfl, rho, T, mom, U_in, U_out);
    if (oned_eligible(g)) return oned_impl(g, dt_device, cfl, rho, T, mom, U_in, U_out);
    int32_t rc = explicit_impl(g, 0.0, dt_device, rho, T, U_in, U_out);
    if (rc != RT_OK) return rc;
    return implicit_impl(g, 0.0, dt_device, rho, T, mom, U_out, true, cfl, dt_device);
}

extern "C" int32_t rt_rk2_step(rt_grid* g, double* dt_device, double cfl, const double* rho, double* T, double* const mom[3],
                               double* const U[4], double* const W1[4], double* const W2[4]) {
    DeviceGuard dg_(g);
    if (!g || !aligned8(dt_device)) return fail(g, RT_ERR_INVALID_ARG, "rt_rk2_step: null or misaligned dt_device");
    if (!(cfl > 0.0) || !isfinite(cfl)) return fail(g, RT_ERR_INVALID_ARG, "rt_rk2_step: cfl must be finite and > 0");
    if (!aligned8(rho) || !aligned8(T) || !U || !W1 || !W2) return fail(g, RT_ERR_INVALID_ARG, "rt_rk2_step: null or misaligned argument");
    if (!g->have_par) return fail(g, RT_ERR_BAD_STATE, "rt_rk2_step: rt_set_params has not been called");
    for (int q = 0; q < 4; ++q)
        if (!aligned8(U[q]) || !aligned8(W1[q]) || !aligned8(W2[q]) || U[q] == W1[q] || U[q] == W2[q] || W1[q] == W2[q])
            return fail(g, RT_ERR_INVALID_ARG, "rt_rk2_step: U/W1/W2[%d] null, misaligned or aliased", q);
    const bool feedback = g->par.feedback_momentum && mom != nullptr;
    if (feedback)
        for (int q = 0; q < 3; ++q)
            if (!aligned8(mom[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_rk2_step: mom[%d] null or misaligned", q);
    const GridDev& D = g->dev;
    const size_t bytes = (size_t)D.ntot * sizeof(double);
    const int nsave = feedback ? 4 : 1;
    for (int q = 0; q < nsave; ++q)
        if (!g->rk_save[q]) RT_CUDA(g, cudaMalloc(&g->rk_save[q], bytes));
    if (!g->rk_dt) RT_CUDA(g, cudaMalloc(&g->rk_dt, 2 * sizeof(double)));
    RT_CUDA(g, cudaMemcpyAsync(g->rk_dt, dt_device, sizeof(double), cudaMemcpyDeviceToDevice, g->stream));
    RT_CUDA(g, cudaMemcpyAsync(g->rk_dt + 1, dt_device, sizeof(double), cudaMemcpyDeviceToDevice, g->stream));
    if (fused_eligible(g) && g->par.solver != RT_SOLVER_RUSANOV) {
        // Both stages in the fused kernel, nothing copied.  Stage 1 reads T^n, m^n and writes T_1, m_1 into the handle's
        // scratch arrays; stage 2 reads those (in place) and stores the averages (U + U_2)/2 into U, (T^n + T_2)/2 into T,
        // (m^n + m_2)/2 into m, and reduces the CFL rate of the AVERAGED state: no save copies, no averaging pass, no
        // separate CFL pass, W2 untouched.
        RkAvg s1;
        memset(&s1, 0, sizeof(s1));
        s1.Tout = g->rk_save[0];
        for (int q = 0; q < 3; ++q) s1.mout[q] = feedback ? g->rk_save[1 + q] : nullptr;
        int32_t rc1 = fused_impl(g, g->rk_dt, cfl, rho, T, mom, U, W1, &s1);
        if (rc1 != RT_OK) return rc1;
        RkAvg s2;
        memset(&s2, 0, sizeof(s2));
        for (int q = 0; q < 4; ++q) s2.U[q] = U[q];
        s2.T = T;
        for (int q = 0; q < 3; ++q) s2.m[q] = feedback ? mom[q] : nullptr;
        s2.Tout = T;
        for (int q = 0; q < 3; ++q) s2.mout[q] = feedback ? mom[q] : nullptr;
        s2.dt_out = dt_device;
        double* m1[3] = {g->rk_save[1], g->rk_save[2], g->rk_save[3]};
        return fused_impl(g, g->rk_dt + 1, cfl, rho, g->rk_save[0], feedback ? m1 : nullptr, W1, U, &s2);
    }
    // T^n, m^n (the sub-steps update them in place)
    RT_CUDA(g, cudaMemcpyAsync(g->rk_save[0], T, bytes, cudaMemcpyDeviceToDevice, g->stream));
    for (int q = 0; q < 3 && feedback; ++q)
        RT_CUDA(g, cudaMemcpyAsync(g->rk_save[1 + q], mom[q], bytes, cudaMemcpyDeviceToDevice, g->stream));
    int32_t rc = substep_impl(g, g->rk_dt, cfl, rho, T, mom, U, W1);
    if (rc != RT_OK) return rc;
    rc = substep_impl(g, g->rk_dt + 1, cfl, rho, T, mom, W1, W2);
    if (rc != RT_OK) return rc;
    AvgArgs v;
    memset(&v, 0, sizeof(v));
    for (int q = 0; q < 4; ++q) {
        v.a[q] = U[q];
        v.b[q] = W2[q];
    }
    v.a[4] = T;                 // T <- (T^n + T^2)/2: a holds T^2 here, b the saved T^n: the average is symmetric
    v.b[4] = g->rk_save[0];
    v.n = 5;
    for (int q = 0; q < 3 && feedback; ++q) {
        v.a[5 + q] = mom[q];
        v.b[5 + q] = g->rk_save[1 + q];
        v.n = 8;
    }
    const int bx = D.n[0] >= 128 ? 128 : ((D.n[0] + 31) / 32) * 32;
    dim3 grid((D.n[0] + bx - 1) / bx, D.n[1], D.n[2]);
    k_rk2_average<<<grid, bx, 0, g->stream>>>(D, v);
    RT_LAUNCH_CHECK(g);
    return rt_cfl_dt_async(g, U, cfl, dt_device);
}

extern "C" int32_t rt_cfl_dt_async(rt_grid* g, const double* const U[4], double cfl, double* dt_device) {
    DeviceGuard dg_(g);
    if (!g || !U || !dt_device) return fail(g, RT_ERR_INVALID_ARG, "rt_cfl_dt: null argument");
    if (!g->have_par) return fail(g, RT_ERR_BAD_STATE, "rt_cfl_dt: rt_set_params has not been called");
    if (!(cfl > 0.0) || !isfinite(cfl)) return fail(g, RT_ERR_INVALID_ARG, "rt_cfl_dt: cfl must be finite and > 0");
    for (int q = 0; q < 4; ++q)
        if (!aligned8(U[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_cfl_dt: U[%d] null or misaligned", q);
    const GridDev& D = g->dev;
    const long long nrows = (long long)D.n[1] * D.n[2];
    const int nb = (int)(nrows < 148 * 8 ? nrows : 148 * 8);
    {
        ProfScope ps(g, RT_K_CFL);
        k_cfl<<<nb, 256, 0, g->stream>>>(D, g->par.chat, U[0], U[1], U[2], U[3], g->scr, cfl, dt_device);
    }
    RT_LAUNCH_CHECK(g);
    return RT_OK;
}

extern "C" int32_t rt_cfl_dt(rt_grid* g, const double* const U[4], double cfl, double* dt_host) {
    DeviceGuard dg_(g);
    if (!dt_host) return fail(g, RT_ERR_INVALID_ARG, "rt_cfl_dt: null argument");
    int32_t rc = rt_cfl_dt_async(g, U, cfl, g ? g->dt_dev : nullptr);
    if (rc != RT_OK) return rc;
    RT_CUDA(g, cudaMemcpyAsync(g->dt_pinned, g->dt_dev, sizeof(double), cudaMemcpyDeviceToHost, g->stream));
    RT_CUDA(g, cudaStreamSynchronize(g->stream));
    *dt_host = *g->dt_pinned;
    return RT_OK;
}

extern "C" int32_t rt_check_finite(rt_grid* g, const double* const U[4], const double* T, int64_t* n_bad) {
    DeviceGuard dg_(g);
    if (!g || !U) return fail(g, RT_ERR_INVALID_ARG, "rt_check_finite: null argument");
    FiniteArgs v;
    memset(&v, 0, sizeof(v));
    for (int q = 0; q < 4; ++q) {
        if (!aligned8(U[q])) return fail(g, RT_ERR_INVALID_ARG, "rt_check_finite: U[%d] null or misaligned", q);
        v.f[q] = U[q];
    }
    v.n = 4;
    if (T) {
        if (!aligned8(T)) return fail(g, RT_ERR_INVALID_ARG, "rt_check_finite: T misaligned");
        v.f[v.n++] = T;
    }
    const GridDev& D = g->dev;
    // the clip counter's word serves as scratch: save it, count, restore
    RT_CUDA(g, cudaMemcpyAsync(g->counters_pinned, g->counters, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, g->stream));
    RT_CUDA(g, cudaMemsetAsync(g->counters + 1, 0, sizeof(unsigned long long), g->stream));
    const int bx = D.n[0] >= 128 ? 128 : ((D.n[0] + 31) / 32) * 32;
    dim3 grid((D.n[0] + bx - 1) / bx, D.n[1], D.n[2]);
    k_check_finite<<<grid, bx, 0, g->stream>>>(D, v, g->counters + 1);
    RT_LAUNCH_CHECK(g);
    unsigned long long saved[2];
    RT_CUDA(g, cudaStreamSynchronize(g->stream));
    saved[0] = g->counters_pinned[0];
    saved[1] = g->counters_pinned[1];
    RT_CUDA(g, cudaMemcpyAsync(g->counters_pinned, g->counters + 1, sizeof(unsigned long long), cudaMemcpyDeviceToHost, g->stream));
    RT_CUDA(g, cudaStreamSynchronize(g->stream));
    const unsigned long long bad = g->counters_pinned[0];
    g->counters_pinned[0] = saved[1];
    RT_CUDA(g, cudaMemcpyAsync(g->counters + 1, g->counters_pinned, sizeof(unsigned long long), cudaMemcpyHostToDevice, g->stream));
    RT_CUDA(g, cudaStreamSynchronize(g->stream));
    if (n_bad) *n_bad = (int64_t)bad;
    if (bad) return fail(g, RT_ERR_NOT_FINITE, "rt_check_finite: %llu interior cells hold a non-finite value", bad);
    return RT_OK;
}

extern "C" int32_t rt_get_floor_counts(rt_grid* g, int64_t* n_floor, int64_t* n_clip) {
    DeviceGuard dg_(g);
    if (!g) return RT_ERR_INVALID_ARG;
    RT_CUDA(g, cudaMemcpyAsync(g->counters_pinned, g->counters, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, g->stream));
    RT_CUDA(g, cudaMemsetAsync(g->counters, 0, 2 * sizeof(unsigned long long), g->stream));
    RT_CUDA(g, cudaStreamSynchronize(g->stream));
    if (n_floor) *n_floor = (int64_t)g->counters_pinned[0];
    if (n_clip) *n_clip = (int64_t)g->counters_pinned[1];
    return RT_OK;
}

// ------------------------------------------------------------------------------------------------
// Measurement hook (no grid handle): time one launch of the DFMA-chain microbenchmark with CUDA events on `cuda_stream`.
extern "C" int32_t rt_measure_fp64(void* cuda_stream, int32_t blocks, int32_t threads, int32_t chains, int32_t iters,
                                   double* ms_host) {
    if (!ms_host || blocks < 1 || threads < 32 || threads > 1024 || (threads & 31) || iters < 1) return RT_ERR_INVALID_ARG;
    if (chains != 1 && chains != 2 && chains != 4 && chains != 8 && chains != 101 && chains != 102 && chains != 104 &&
        chains != 204 && chains != 304 && chains != 214 && chains != 314)
        return RT_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    double* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int32_t rc = RT_ERR_CUDA;
    if (cudaMalloc(&sink, sizeof(double)) == cudaSuccess && cudaEventCreate(&e0) == cudaSuccess &&
        cudaEventCreate(&e1) == cudaSuccess) {
        const double a = 0.999999, b = 1.0e-6;  // x -> 1: finite for any iteration count
        for (int pass = 0; pass < 2; ++pass) {  // pass 0 warms up (module load, clocks)
            cudaEventRecord(e0, st);
            switch (chains) {
                case 1: k_dfma_chains<1><<<blocks, threads, 0, st>>>(sink, iters, a, b); break;
                case 2: k_dfma_chains<2><<<blocks, threads, 0, st>>>(sink, iters, a, b); break;
                case 4: k_dfma_chains<4><<<blocks, threads, 0, st>>>(sink, iters, a, b); break;
                case 101: k_dfma_chains<1, 64><<<blocks, threads, 0, st>>>(sink, iters, a, b); break;
                case 102: k_dfma_chains<2, 64><<<blocks, threads, 0, st>>>(sink, iters, a, b); break;
                case 104: k_dfma_chains<4, 64><<<blocks, threads, 0, st>>>(sink, iters, a, b); break;
                case 204: k_dfma_operands<2, 0><<<blocks, threads, 0, st>>>(sink, iters, a, b, 1.0f, 0.0f); break;
                case 304: k_dfma_operands<3, 0><<<blocks, threads, 0, st>>>(sink, iters, a, b, 1.0f, 0.0f); break;
                case 214: k_dfma_operands<2, 4><<<blocks, threads, 0, st>>>(sink, iters, a, b, 1.0f, 0.0f); break;
                case 314: k_dfma_operands<3, 4><<<blocks, threads, 0, st>>>(sink, iters, a, b, 1.0f, 0.0f); break;
                default: k_dfma_chains<8><<<blocks, threads, 0, st>>>(sink, iters, a, b); break;
            }
            cudaEventRecord(e1, st);
        }
        float t = 0.f;
        if (cudaGetLastError() == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess &&
            cudaEventElapsedTime(&t, e0, e1) == cudaSuccess) {
            *ms_host = (double)t;
            rc = RT_OK;
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    return rc;
}
