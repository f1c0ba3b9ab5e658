// gdn_api.cu -- the C ABI of include/gdn.h: plan / forward / destroy.
// Host logic only (validation, path choice, workspace, launches); every arithmetic step of the path
// runs in the kernels of gdn_simt.cuh (fp32 CUDA cores) and gdn_tc_*.cuh (tcgen05 tensor cores).
#include "../../include/gdn.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "gdn_frontend.cuh"
#include "gdn_profile.cuh"
#include "gdn_simt.cuh"
#include "gdn_tc.cuh"

struct gdn_plan;

namespace {

thread_local std::string g_plan_error;

// ---------------------------------------------------------------------------------------------------
// gdn_compute_gates_static (include/gdn.h): the gates of Eq. 13-15 with NO allocation of any kind.  Its scratch (the partial
// frame sums of W_alpha . x_n and the per-frame arrival counters that gdn_compute_gates keeps in a plan-owned cudaMalloc'd
// buffer) lives in this file-scope device array: every GPU that loads the library holds these 80 KB until the process exits,
// and every call on a device shares them.  In HOST code the array's name is a host-side stand-in, not a device address: the
// launch below passes the address cudaGetSymbolAddress returns for the current device (looked up once per device).
// ---------------------------------------------------------------------------------------------------
constexpr int kStaticGateMaxFrames = 4096;      // B * H * (T / group) at most
constexpr int kStaticGateMaxParts = 16384;      // B * H * (T / group) * (token splits per frame) at most
static __device__ __align__(256) unsigned int g_gates_static_scratch[kStaticGateMaxParts + kStaticGateMaxFrames];   // partial sums (fp32) | counters

__global__ void __launch_bounds__(gdn::fe::kFeThreads, 4)
gdn_gates_static_kernel(const gdn::GateParams gp) {
    __shared__ float s_sum[16];
    __shared__ unsigned int s_last;
    gdn::fe::gates_body(gp, (int)blockIdx.x / gp.NSPL, (int)blockIdx.x % gp.NSPL, s_sum, &s_last);
}

// gdn_forward_chunk_host: device staging plus a copy/compute pipeline over token segments.  The call is cut into
// up to kMaxSeg segments of Tseg tokens (whole 128-token tiles, resp. whole frames; exact by the split invariance of
// the recurrence, PAPER.md L72 / App. G.6): segment s+1 travels host->device on a copy stream while segment s is
// computed on the caller's stream and the output of segment s-1 travels back on a second copy stream.
constexpr int kMaxSeg = 8;
struct Staging {
    void *q = nullptr, *k = nullptr, *v = nullptr, *out = nullptr;     // per segment compact [B,Tseg,H,d]
    float *alpha = nullptr, *beta = nullptr, *state = nullptr;          // per segment compact [B,H,Tseg/G], [B,H,Tseg]
    bool ready = false;
    int nseg = 1, Tseg = 0, Ttail = 0;           // nseg-1 segments of Tseg tokens, then one of Ttail (== Tseg if it divides)
    gdn_plan_t* seg_plan = nullptr;               // plan for T = Tseg (nullptr: the owning plan itself, nseg == 1)
    gdn_plan_t* tail_plan = nullptr;               // plan for T = Ttail when Ttail != Tseg
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_out = nullptr, ev_in[kMaxSeg] = {}, ev_comp[kMaxSeg] = {};
    // unsegmented calls (nseg == 1): a second set of input staging buffers, so that the inputs of call i+1 travel on the copy-in
    // stream while call i computes and copies out (ev_in[par] / ev_comp[par] are used per parity)
    void *q2 = nullptr, *k2 = nullptr, *v2 = nullptr;
    float *alpha2 = nullptr, *beta2 = nullptr;
    unsigned long long calls = 0;
    const void* prev_out_lo[2] = {nullptr, nullptr};   // host ranges the previous call writes: [out_host), [state_out_host)
    const void* prev_out_hi[2] = {nullptr, nullptr};
};

}  // namespace

namespace {
// release everything the host entry point set up (also after a partial set-up, so that a retry starts clean)
void staging_free(Staging& h) {
    void* bufs[] = {h.q, h.k, h.v, h.out, h.alpha, h.beta, h.state, h.q2, h.k2, h.v2, h.alpha2, h.beta2};
    for (void* b : bufs) if (b) cudaFree(b);
    h.q = h.k = h.v = h.out = nullptr; h.alpha = h.beta = h.state = nullptr;
    h.q2 = h.k2 = h.v2 = nullptr; h.alpha2 = h.beta2 = nullptr;
    h.calls = 0;
    if (h.seg_plan) gdn_destroy(h.seg_plan);
    if (h.tail_plan) gdn_destroy(h.tail_plan);
    h.seg_plan = h.tail_plan = nullptr;
    if (h.s_in) cudaStreamDestroy(h.s_in);
    if (h.s_out) cudaStreamDestroy(h.s_out);
    h.s_in = h.s_out = nullptr;
    if (h.ev_start) cudaEventDestroy(h.ev_start);
    if (h.ev_out) cudaEventDestroy(h.ev_out);
    h.ev_start = h.ev_out = nullptr;
    for (int i = 0; i < kMaxSeg; ++i) {
        if (h.ev_in[i]) cudaEventDestroy(h.ev_in[i]);
        if (h.ev_comp[i]) cudaEventDestroy(h.ev_comp[i]);
        h.ev_in[i] = h.ev_comp[i] = nullptr;
    }
    h.ready = false;
}
}  // namespace

struct gdn_plan {
    gdn_config_t cfg;
    int device = -1;
    int sm_count = 0;
    int cc_major = 0, cc_minor = 0;
    gdn_path_t path = GDN_PATH_SIMT_FP32;
    int chunk = 0;
    int launches = 1;
    void* workspace = nullptr;
    size_t workspace_bytes = 0;
    float* z_stage = nullptr;     // copy of z_in when z_out aliases it
    // front end (gdn_feature_map / gdn_compute_gates / gdn_forward_chunk_full), allocated at first use
    void* fe_feat = nullptr;      // q_rot | k_rot | q_raw | k_raw, dense [B,T,H,D] bf16 each
    float* fe_gates = nullptr;    // alpha [B,H,F] | beta [B,H,T] | partial frame sums | counters
    int fe_nspl = 1;
    // CUDA graphs of the multi-launch frame-wise calls, one per tuple of argument pointers (see run_graphed)
    struct GraphEntry { std::vector<const void*> key; cudaGraphExec_t exec = nullptr; unsigned long long used = 0; };
    std::vector<GraphEntry> graphs;
    unsigned long long graph_tick = 0;
    bool graph_warm = false;      // the first call of a plan is issued directly (kernel attributes, lazy allocations)
    Staging host;
    gdn::TcPlan tc;               // tensor-core path state (tensor maps, workspace carving)
    gdn::Profiler prof;           // optional per-kernel CUDA events (bench roofline)
    std::string err;
};

namespace {

size_t esize(int dt) { return dt == GDN_FP32 ? 4 : 2; }

bool head_dim_ok(int d) { return d == 32 || d == 64 || d == 128; }

gdn_status_t fail(gdn_plan_t* p, gdn_status_t st, const std::string& msg) {
    if (p) p->err = msg; else g_plan_error = msg;
    return st;
}

gdn_status_t cuda_fail(gdn_plan_t* p, cudaError_t e, const char* what) {
    return fail(p, GDN_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

long long tok_stride(long long s, int H, int d) { return s ? s : (long long)H * d; }

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <typename TIn>
void launch_simt(const gdn::SimtParams& sp, int dk, cudaStream_t st) {
    const int tiles = sp.dv / gdn::kSimtCols;
    const long long warps = (long long)sp.B * sp.H * tiles;
    const int blocks = (int)((warps + gdn::kSimtWarps - 1) / gdn::kSimtWarps);
    const dim3 block(gdn::kSimtWarps * 32);
    switch (dk) {
        case 32:  gdn::gdn_simt_kernel<32, TIn><<<blocks, block, 0, st>>>(sp); break;
        case 64:  gdn::gdn_simt_kernel<64, TIn><<<blocks, block, 0, st>>>(sp); break;
        default:  gdn::gdn_simt_kernel<128, TIn><<<blocks, block, 0, st>>>(sp); break;
    }
}

gdn_status_t check_device(gdn_plan_t* p) {
    if (p->device < 0) return fail(p, GDN_ERR_CUDA, "no CUDA device was visible when the plan was created");
    if (!(p->cc_major == 10 && p->cc_minor == 0))
        return fail(p, GDN_ERR_ARCH, "device is sm_" + std::to_string(p->cc_major * 10 + p->cc_minor) +
                                         ", this library only carries sm_100a code (no fallback)");
    return GDN_OK;
}

gdn_status_t forward_impl(gdn_plan_t* p, const void* q, const void* k, const void* v,
                          const void* q_raw, const void* k_raw,
                          const float* alpha, const float* beta, const float* S_in, const float* z_in,
                          void* out, float* S_out, float* z_out, cudaStream_t st, bool normalizer,
                          const void* out_gate = nullptr, bool dense_qk = false) {
    const gdn_config_t& c = p->cfg;
    const size_t state_elems = (size_t)c.B * c.H * c.d_k * c.d_v;
    if (c.B == 0 || c.H == 0) return GDN_OK;
    if (!S_out) return fail(p, GDN_ERR_INVALID_ARG, "state_out is NULL");
    if (c.T == 0) {                                   // empty chunk: the state passes through
        gdn_status_t ds = check_device(p);
        if (ds != GDN_OK) return ds;
        cudaError_t e = cudaSuccess;
        if (S_in == nullptr) e = cudaMemsetAsync(S_out, 0, state_elems * 4, st);
        else if (S_in != S_out) e = cudaMemcpyAsync(S_out, S_in, state_elems * 4, cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess && normalizer && z_out) {
            if (z_in == nullptr) e = cudaMemsetAsync(z_out, 0, (size_t)c.B * c.H * c.d_k * 4, st);
            else if (z_in != z_out) e = cudaMemcpyAsync(z_out, z_in, (size_t)c.B * c.H * c.d_k * 4, cudaMemcpyDeviceToDevice, st);
        }
        return e == cudaSuccess ? GDN_OK : cuda_fail(p, e, "state pass-through");
    }
    if (!q || !k || !v || !alpha || !beta || !out)
        return fail(p, GDN_ERR_INVALID_ARG, "a required tensor pointer is NULL");
    if (normalizer && (!q_raw || !k_raw || !z_out))
        return fail(p, GDN_ERR_INVALID_ARG, "normaliser call needs q_raw, k_raw and z_out");
    const void* ptrs[] = {q, k, v, alpha, beta, S_in, out, S_out, q_raw, k_raw, z_in, z_out};
    for (const void* ptr : ptrs)
        if (ptr && !aligned16(ptr)) return fail(p, GDN_ERR_ALIGNMENT, "tensor pointers must be 16-byte aligned");
    if (out == q || out == k || out == v) return fail(p, GDN_ERR_INVALID_ARG, "out must not alias an input");
    gdn_status_t ds = check_device(p);
    if (ds != GDN_OK) return ds;
    {   // a plan is bound to the device it was created on (workspace, tensor maps, kernel attributes)
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess || cur != p->device)
            return fail(p, GDN_ERR_INVALID_ARG, "the current device is not the one the plan was created on (device " + std::to_string(p->device) + ")");
    }

    if (p->path != GDN_PATH_SIMT_FP32) {
        std::string msg;
        gdn::NormArgs na{q_raw, k_raw, z_in, z_out};
        na.gate = out_gate; na.g_ts = c.o_token_stride; na.dense_qk = dense_qk;
        gdn_status_t ts = gdn::tc_forward(p->tc, c, q, k, v, alpha, beta, S_in, out, S_out, st, &p->prof, &msg, normalizer ? &na : nullptr);
        if (ts != GDN_OK) return fail(p, ts, msg);
        return GDN_OK;
    }

    if (normalizer && z_in && z_in == z_out) {        // every column tile reads z_in: stage a copy
        cudaError_t e = cudaMemcpyAsync(p->z_stage, z_in, (size_t)c.B * c.H * c.d_k * 4, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return cuda_fail(p, e, "z staging copy");
        z_in = p->z_stage;
    }
    gdn::SimtParams sp{};
    sp.q = q; sp.k = k; sp.v = v; sp.q_raw = q_raw; sp.k_raw = k_raw;
    sp.alpha = alpha; sp.beta = beta; sp.S_in = S_in; sp.z_in = z_in;
    sp.out = out; sp.S_out = S_out; sp.z_out = z_out;
    sp.B = c.B; sp.H = c.H; sp.T = c.T; sp.G = c.group; sp.dv = c.d_v;
    sp.q_ts = tok_stride(c.q_token_stride, c.H, c.d_k);
    sp.k_ts = tok_stride(c.k_token_stride, c.H, c.d_k);
    sp.v_ts = tok_stride(c.v_token_stride, c.H, c.d_v);
    sp.o_ts = tok_stride(c.o_token_stride, c.H, c.d_v);
    sp.scale = c.scale; sp.eps = c.eps;
    sp.log_alpha = (c.flags & GDN_FLAG_LOG_ALPHA) ? 1 : 0;
    sp.normalizer = normalizer ? 1 : 0;
    p->prof.begin(st);
    if (c.io_dtype == GDN_FP32) launch_simt<float>(sp, c.d_k, st);
    else launch_simt<__nv_bfloat16>(sp, c.d_k, st);
    p->prof.mark(st, "gdn_simt_kernel");
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e, "gdn_simt_kernel launch");
    return GDN_OK;
}



// The frame-wise paths are three to five launches per call (two streams where the normaliser runs as a pass of its own); at the paper's production chunk (8 MB of
// input) the host cannot issue them as fast as the GPU retires them.  So a call is captured ONCE per tuple of argument
// pointers into a CUDA graph (fork / join with the normaliser's stream and the programmatic launch edges included) and
// replayed afterwards: one graph launch per call.  Not used when per-kernel profiling is on, when the caller is itself
// capturing `st` (the launches then simply go into the caller's graph), or on the legacy default stream.
constexpr size_t kMaxGraphs = 32;
template <typename Issue>
gdn_status_t run_graphed(gdn_plan_t* p, std::vector<const void*> key, cudaStream_t st, Issue&& issue) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (p->prof.enabled() || st == nullptr || cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        return issue();
    }
    if (!p->graph_warm) { p->graph_warm = true; return issue(); }
    for (auto& g : p->graphs)
        if (g.key == key) {
            g.used = ++p->graph_tick;
            cudaError_t e = cudaGraphLaunch(g.exec, st);
            return e == cudaSuccess ? GDN_OK : cuda_fail(p, e, "graph launch");
        }
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return issue(); }
    const gdn_status_t is = issue();
    cudaGraph_t graph = nullptr;
    const cudaError_t ee = cudaStreamEndCapture(st, &graph);
    if (is != GDN_OK) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return is; }
    if (ee != cudaSuccess || !graph) { cudaGetLastError(); return issue(); }       // not capturable here: issue directly
    cudaGraphExec_t exec = nullptr;
    const cudaError_t ie = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ie != cudaSuccess || !exec) { cudaGetLastError(); return issue(); }
    if (p->graphs.size() >= kMaxGraphs) {                                            // evict the least recently used
        size_t lru = 0;
        for (size_t i = 1; i < p->graphs.size(); ++i) if (p->graphs[i].used < p->graphs[lru].used) lru = i;
        cudaGraphExecDestroy(p->graphs[lru].exec);
        p->graphs.erase(p->graphs.begin() + (long)lru);
    }
    gdn_plan::GraphEntry ge;
    ge.key = std::move(key); ge.exec = exec; ge.used = ++p->graph_tick;
    p->graphs.push_back(std::move(ge));
    const cudaError_t le = cudaGraphLaunch(exec, st);
    return le == cudaSuccess ? GDN_OK : cuda_fail(p, le, "graph launch");
}

inline uint32_t __float_as_uint_host(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

bool graphable(const gdn_plan_t* p) { return p->path == GDN_PATH_TC_FRAME && p->cfg.T > 0 && p->cfg.B > 0 && p->cfg.H > 0; }

// ---- front end ----------------------------------------------------------------------------------------
gdn_status_t fe_check(gdn_plan_t* p) {
    const gdn_config_t& c = p->cfg;
    if (c.io_dtype != GDN_BF16 || c.d_k != c.d_v || c.d_k % 8 != 0 || c.d_k > 128)
        return fail(p, GDN_ERR_UNSUPPORTED, "the front end needs a bf16 plan with d_k = d_v a multiple of 8, at most 128");
    if ((long long)c.B * c.T * c.H >= (1LL << 31) - 64 * 1024)
        return fail(p, GDN_ERR_UNSUPPORTED, "the front end indexes (token, head) rows with 32 bits: B*T*H must stay below 2^31");
    gdn_status_t ds = check_device(p);
    if (ds != GDN_OK) return ds;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != p->device)
        return fail(p, GDN_ERR_INVALID_ARG, "the current device is not the one the plan was created on");
    return GDN_OK;
}

// validate + fill; returns GDN_OK with `active` = false for an empty problem
gdn_status_t featmap_fill(gdn_plan_t* p, const gdn_featmap_args_t* a, void* q_rot, void* k_rot, void* q_raw, void* k_raw,
                          gdn::FeatmapParams& fp, bool& active) {
    const gdn_config_t& c = p->cfg;
    active = false;
    if (!a || !a->q || !a->k || !a->rms_wq || !a->rms_wk || !a->rope_cos || !a->rope_sin || !q_rot || !k_rot || !q_raw || !k_raw)
        return fail(p, GDN_ERR_INVALID_ARG, "a required feature-map pointer is NULL");
    const void* ptrs[] = {a->q, a->k, a->rms_wq, a->rms_wk, a->rope_cos, a->rope_sin, q_rot, k_rot, q_raw, k_raw};
    for (const void* ptr : ptrs) if (!aligned16(ptr)) return fail(p, GDN_ERR_ALIGNMENT, "tensor pointers must be 16-byte aligned");
    if (c.B == 0 || c.H == 0 || c.T == 0) return GDN_OK;
    fp = gdn::FeatmapParams{};
    fp.q = static_cast<const __nv_bfloat16*>(a->q); fp.k = static_cast<const __nv_bfloat16*>(a->k);
    fp.wq = a->rms_wq; fp.wk = a->rms_wk; fp.cosT = a->rope_cos; fp.sinT = a->rope_sin;
    fp.q_rot = static_cast<__nv_bfloat16*>(q_rot); fp.k_rot = static_cast<__nv_bfloat16*>(k_rot);
    fp.q_raw = static_cast<__nv_bfloat16*>(q_raw); fp.k_raw = static_cast<__nv_bfloat16*>(k_raw);
    fp.q_ts = tok_stride(c.q_token_stride, c.H, c.d_k); fp.k_ts = tok_stride(c.k_token_stride, c.H, c.d_k);
    fp.B = c.B; fp.T = c.T; fp.H = c.H; fp.D = c.d_k;
    fp.rms_eps = a->rms_eps;
    fp.kscale = 1.f / sqrtf((float)c.d_k * (float)c.group);
    active = true;
    return GDN_OK;
}

size_t fe_up4(size_t n) { return (n + 3) / 4 * 4; }        // 16-byte aligned sub-buffers

gdn_status_t fe_gate_buffers(gdn_plan_t* p) {
    if (p->fe_gates) return GDN_OK;
    const gdn_config_t& c = p->cfg;
    const size_t BH = (size_t)c.B * c.H, F = (size_t)(c.T / c.group);
    // splits per frame: enough CTAs to fill the GPU, at least 64 tokens each
    int nspl = (int)((4 * (size_t)(p->sm_count > 0 ? p->sm_count : 148) + BH * F - 1) / (BH * F));
    const int max_spl = (c.group + 63) / 64;
    if (nspl > max_spl) nspl = max_spl;
    if (nspl < 1) nspl = 1;
    p->fe_nspl = nspl;
    const size_t words = fe_up4(BH * F) + fe_up4(BH * c.T) + BH * F * nspl + BH * F;      // alpha | beta | partials | counters
    if (cudaMalloc(&p->fe_gates, words * 4) != cudaSuccess) { cudaGetLastError(); return fail(p, GDN_ERR_NOMEM, "gate buffer allocation failed"); }
    if (cudaMemset(p->fe_gates, 0, words * 4) != cudaSuccess) { cudaGetLastError(); return fail(p, GDN_ERR_CUDA, "gate buffer initialisation failed"); }
    return GDN_OK;
}

gdn_status_t gates_fill(gdn_plan_t* p, const gdn_gate_args_t* a, float* alpha_out, float* beta_out, gdn::GateParams& gp, bool& active) {
    const gdn_config_t& c = p->cfg;
    active = false;
    if (!a || !a->x || !a->w_alpha || !a->b_alpha || !a->a_log || !a->w_beta || !a->b_beta || !alpha_out || !beta_out)
        return fail(p, GDN_ERR_INVALID_ARG, "a required gate pointer is NULL");
    if (!aligned16(a->x) || (a->x_token_stride % 8) != 0) return fail(p, GDN_ERR_ALIGNMENT, "x must be 16-byte aligned with a token stride that is a multiple of 8");
    if (c.B == 0 || c.H == 0 || c.T == 0) return GDN_OK;
    gdn_status_t bs = fe_gate_buffers(p);
    if (bs != GDN_OK) return bs;
    const size_t BH = (size_t)c.B * c.H, F = (size_t)(c.T / c.group);
    gp = gdn::GateParams{};
    gp.x = static_cast<const __nv_bfloat16*>(a->x);
    gp.w_alpha = a->w_alpha; gp.b_alpha = a->b_alpha; gp.a_log = a->a_log; gp.w_beta = a->w_beta; gp.b_beta = a->b_beta;
    gp.alpha_out = alpha_out; gp.beta_out = beta_out;
    gp.part = p->fe_gates + fe_up4(BH * F) + fe_up4(BH * c.T);
    gp.counters = reinterpret_cast<unsigned int*>(gp.part + BH * F * p->fe_nspl);
    gp.x_ts = tok_stride(a->x_token_stride, c.H, c.d_k);
    gp.B = c.B; gp.T = c.T; gp.H = c.H; gp.D = c.d_k; gp.G = c.group; gp.F = (int)F; gp.NSPL = p->fe_nspl;
    gp.log_alpha = (c.flags & GDN_FLAG_LOG_ALPHA) ? 1 : 0;
    active = true;
    return GDN_OK;
}

// ONE launch for whichever parts are active: B*H*F*NSPL gate blocks, then the feature-map blocks
gdn_status_t launch_frontend(gdn_plan_t* p, const gdn::FeatmapParams* fm, const gdn::GateParams* gp, cudaStream_t st, bool mark) {
    int n_fm = 0, n_g = 0;
    if (fm) {
        const long long rows = (long long)fm->B * fm->T * fm->H, per = 16LL * gdn::fe::kFeRows;
        long long blocks = (rows + per - 1) / per;
        const long long cap = 8LL * (p->sm_count > 0 ? p->sm_count : 148);
        n_fm = (int)(blocks > cap ? cap : blocks);
    }
    if (gp) n_g = gp->B * gp->H * gp->F * gp->NSPL;
    if (n_fm + n_g == 0) return GDN_OK;
    gdn::GateParams g0{};
    g0.NSPL = 1;
    gdn::fe::gdn_frontend_kernel<<<n_fm + n_g, gdn::fe::kFeThreads, 0, st>>>(fm ? *fm : gdn::FeatmapParams{}, gp ? *gp : g0, n_g);
    if (mark) p->prof.mark(st, "gdn_frontend_kernel");
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? GDN_OK : cuda_fail(p, e, "gdn_frontend_kernel launch");
}

}  // namespace

extern "C" {

gdn_status_t gdn_plan(const gdn_config_t* cfg, gdn_plan_t** plan_out) {
    if (plan_out) *plan_out = nullptr;
    if (!cfg || !plan_out) return fail(nullptr, GDN_ERR_INVALID_ARG, "cfg or plan_out is NULL");
    if (cfg->struct_size != sizeof(gdn_config_t))
        return fail(nullptr, GDN_ERR_INVALID_ARG, "struct_size does not match this library's gdn_config_t");
    const gdn_config_t& c = *cfg;
    if (c.B < 0 || c.H < 0 || c.T < 0) return fail(nullptr, GDN_ERR_INVALID_ARG, "B, H, T must be >= 0");
    if (c.d_k <= 0 || c.d_v <= 0 || c.group <= 0) return fail(nullptr, GDN_ERR_INVALID_ARG, "d_k, d_v, group must be > 0");
    if (c.T % c.group != 0) return fail(nullptr, GDN_ERR_INVALID_ARG, "T must be a multiple of group");
    if (c.io_dtype != GDN_BF16 && c.io_dtype != GDN_FP32) return fail(nullptr, GDN_ERR_INVALID_ARG, "unknown io_dtype");
    if (!(c.chunk == 0 || c.chunk == 64 || c.chunk == 128)) return fail(nullptr, GDN_ERR_INVALID_ARG, "chunk must be 0, 64 or 128");
    const uint32_t known = GDN_FLAG_NORMALIZER | GDN_FLAG_BIDIR | GDN_FLAG_LOG_ALPHA | GDN_FLAG_FORCE_SIMT | GDN_FLAG_UNFUSED;
    if (c.flags & ~known) return fail(nullptr, GDN_ERR_INVALID_ARG, "unknown flag bits");
    const bool d112 = c.d_k == 112 && c.d_v == 112;     // the paper's head dim, zero-padded to 128 inside the tensor-core kernels
    if (d112) {
        gdn_path_t pth; int ch = 0, ln = 0;
        if ((c.flags & GDN_FLAG_FORCE_SIMT) || ((c.flags & GDN_FLAG_NORMALIZER) && c.group == 1) || !gdn::tc_supported(c, &pth, &ch, &ln))
            return fail(nullptr, GDN_ERR_UNSUPPORTED, "d = 112 needs a bf16 tensor-core plan (frame-wise, or token-wise with the fused kernel)");
    } else if (!head_dim_ok(c.d_k) || !head_dim_ok(c.d_v))
        return fail(nullptr, GDN_ERR_UNSUPPORTED, "d_k and d_v must each be 32, 64 or 128 (or both 112)");
    // the bidirectional in-chunk scan exists on the frame-wise tensor-core path only (the paper's case, Alg. 1)
    if ((c.flags & GDN_FLAG_BIDIR) && !(c.group > 1 && c.io_dtype == GDN_BF16 && c.d_k == c.d_v && (c.d_k == 64 || c.d_k == 112 || c.d_k == 128) &&
                                        !(c.flags & GDN_FLAG_FORCE_SIMT)))
        return fail(nullptr, GDN_ERR_UNSUPPORTED, "GDN_FLAG_BIDIR needs a frame-wise (group > 1) bf16 plan with d_k = d_v in {64,128}");
    const long long strides[4] = {c.q_token_stride, c.k_token_stride, c.v_token_stride, c.o_token_stride};
    const int dims[4] = {c.d_k, c.d_k, c.d_v, c.d_v};
    for (int i = 0; i < 4; ++i) {
        if (strides[i] < 0) return fail(nullptr, GDN_ERR_INVALID_ARG, "token strides must be >= 0");
        if (strides[i] != 0 && strides[i] < (long long)c.H * dims[i])
            return fail(nullptr, GDN_ERR_INVALID_ARG, "token stride smaller than H*d");
        if (strides[i] % 8 != 0) return fail(nullptr, GDN_ERR_ALIGNMENT, "token strides must be multiples of 8 elements");
    }

    gdn_plan_t* p = new (std::nothrow) gdn_plan_t();
    if (!p) return fail(nullptr, GDN_ERR_NOMEM, "host allocation failed");
    p->cfg = c;
    int dev = -1;
    if (cudaGetDevice(&dev) == cudaSuccess) {
        p->device = dev;
        cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&p->cc_major, cudaDevAttrComputeCapabilityMajor, dev);
        cudaDeviceGetAttribute(&p->cc_minor, cudaDevAttrComputeCapabilityMinor, dev);
    } else {
        cudaGetLastError();          // clear "no device": validation-only plan
    }

    // ---- path choice -----------------------------------------------------------------------------
    p->path = GDN_PATH_SIMT_FP32;
    p->chunk = 0;
    p->launches = 1;
    // the normalised readout has a tensor-core path in the frame-wise form only (the paper's case)
    const bool want_tc = c.io_dtype == GDN_BF16 && !(c.flags & GDN_FLAG_FORCE_SIMT) &&
                         !((c.flags & GDN_FLAG_NORMALIZER) && c.group == 1) && c.B > 0 && c.H > 0 && c.T > 0;
    if (want_tc) {
        std::string msg;
        gdn_path_t path;
        int chunk = 0, launches = 1;
        if (gdn::tc_supported(c, &path, &chunk, &launches)) {
            if (p->device >= 0 && p->cc_major == 10 && p->cc_minor == 0) {
                gdn_status_t ts = gdn::tc_plan_init(p->tc, c, p->sm_count, &msg);
                if (ts != GDN_OK) { gdn::tc_plan_free(p->tc); delete p; return fail(nullptr, ts, msg); }
            }
            // frame path with the normaliser: Phase A and the scan run twice (matrix and z pass), the readout once; at d = 128
            // without a token split one launch does Phase A of both passes and one launch their scans
            p->path = path; p->chunk = chunk; p->launches = (path == GDN_PATH_TC_FRAME && (c.flags & GDN_FLAG_NORMALIZER)) ? ((p->tc.D == 128 && p->tc.NSPLIT == 1) ? launches : 2 * launches - 1) : launches;
            p->workspace_bytes = p->tc.workspace_bytes;
        }
    }
    if ((c.flags & GDN_FLAG_NORMALIZER) && p->device >= 0 && c.B * c.H > 0) {
        cudaError_t e = cudaMalloc(&p->z_stage, (size_t)c.B * c.H * c.d_k * 4);
        if (e != cudaSuccess) { cudaGetLastError(); gdn::tc_plan_free(p->tc); delete p; return fail(nullptr, GDN_ERR_NOMEM, "z staging allocation failed"); }
        p->workspace_bytes += (size_t)c.B * c.H * c.d_k * 4;
    }
    *plan_out = p;
    return GDN_OK;
}

gdn_status_t gdn_forward_chunk(gdn_plan_t* plan, const void* q, const void* k, const void* v,
                               const float* alpha, const float* beta, const float* state_in,
                               void* out, float* state_out, gdn_stream_t stream) {
    if (!plan) return fail(nullptr, GDN_ERR_INVALID_ARG, "plan is NULL");
    if (plan->cfg.flags & GDN_FLAG_NORMALIZER)
        return fail(plan, GDN_ERR_INVALID_ARG, "plan carries GDN_FLAG_NORMALIZER: call gdn_forward_chunk_norm");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    auto issue = [&]() { return forward_impl(plan, q, k, v, nullptr, nullptr, alpha, beta, state_in, nullptr, out, state_out, nullptr, st, false); };
    if (!graphable(plan)) return issue();
    return run_graphed(plan, {(const void*)1, q, k, v, alpha, beta, state_in, out, state_out}, st, issue);
}

gdn_status_t gdn_forward_chunk_norm(gdn_plan_t* plan, const void* q_rot, const void* k_rot, const void* v,
                                    const void* q_raw, const void* k_raw, const float* alpha, const float* beta,
                                    const float* S_in, const float* z_in, void* out, float* S_out, float* z_out,
                                    gdn_stream_t stream) {
    if (!plan) return fail(nullptr, GDN_ERR_INVALID_ARG, "plan is NULL");
    if (!(plan->cfg.flags & GDN_FLAG_NORMALIZER))
        return fail(plan, GDN_ERR_INVALID_ARG, "plan was not created with GDN_FLAG_NORMALIZER");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    auto issue = [&]() { return forward_impl(plan, q_rot, k_rot, v, q_raw, k_raw, alpha, beta, S_in, z_in, out, S_out, z_out, st, true); };
    if (!graphable(plan)) return issue();
    return run_graphed(plan, {(const void*)2, q_rot, k_rot, v, q_raw, k_raw, alpha, beta, S_in, z_in, out, S_out, z_out}, st, issue);
}


gdn_status_t gdn_feature_map(gdn_plan_t* plan, const gdn_featmap_args_t* args, void* q_rot, void* k_rot, void* q_raw, void* k_raw,
                             gdn_stream_t stream) {
    if (!plan) return fail(nullptr, GDN_ERR_INVALID_ARG, "plan is NULL");
    gdn_status_t s = fe_check(plan);
    if (s != GDN_OK) return s;
    gdn::FeatmapParams fp;
    bool on = false;
    s = featmap_fill(plan, args, q_rot, k_rot, q_raw, k_raw, fp, on);
    if (s != GDN_OK || !on) return s;
    plan->prof.begin(static_cast<cudaStream_t>(stream));
    return launch_frontend(plan, &fp, nullptr, static_cast<cudaStream_t>(stream), true);
}

gdn_status_t gdn_compute_gates(gdn_plan_t* plan, const gdn_gate_args_t* args, float* alpha_out, float* beta_out, gdn_stream_t stream) {
    if (!plan) return fail(nullptr, GDN_ERR_INVALID_ARG, "plan is NULL");
    gdn_status_t s = fe_check(plan);
    if (s != GDN_OK) return s;
    gdn::GateParams gp;
    bool on = false;
    s = gates_fill(plan, args, alpha_out, beta_out, gp, on);
    if (s != GDN_OK || !on) return s;
    plan->prof.begin(static_cast<cudaStream_t>(stream));
    return launch_frontend(plan, nullptr, &gp, static_cast<cudaStream_t>(stream), true);
}

gdn_status_t gdn_compute_gates_static(const gdn_gate_args_t* a, int B, int T, int H, int D, int group, int log_alpha,
                                      float* alpha_out, float* beta_out, gdn_stream_t stream) {
    if (B < 0 || H < 0 || T < 0) return fail(nullptr, GDN_ERR_INVALID_ARG, "B, H, T must be >= 0");
    if (group <= 0 || T % group != 0) return fail(nullptr, GDN_ERR_INVALID_ARG, "group must be > 0 and divide T");
    if (D < 8 || D > 128 || D % 8 != 0) return fail(nullptr, GDN_ERR_UNSUPPORTED, "D must be a multiple of 8 between 8 and 128");
    if (!a || !a->x || !a->w_alpha || !a->b_alpha || !a->a_log || !a->w_beta || !a->b_beta || !alpha_out || !beta_out)
        return fail(nullptr, GDN_ERR_INVALID_ARG, "a required gate pointer is NULL");
    if (!aligned16(a->x) || (a->x_token_stride % 8) != 0)
        return fail(nullptr, GDN_ERR_ALIGNMENT, "x must be 16-byte aligned with a token stride that is a multiple of 8");
    if (a->x_token_stride < 0 || (a->x_token_stride != 0 && a->x_token_stride < (long long)H * D))
        return fail(nullptr, GDN_ERR_INVALID_ARG, "x token stride smaller than H*D");
    if (B == 0 || H == 0 || T == 0) return GDN_OK;
    const long long BH = (long long)B * H, F = T / group;
    if (BH * F > kStaticGateMaxFrames)
        return fail(nullptr, GDN_ERR_UNSUPPORTED, "gdn_compute_gates_static: B*H*(T/group) = " + std::to_string(BH * F) +
                                                  " exceeds the static scratch (at most 4096 frame-heads per call); use gdn_compute_gates");
    if (BH * T >= (1LL << 31)) return fail(nullptr, GDN_ERR_UNSUPPORTED, "B*T*H must stay below 2^31");

    // once per device, with that device current: the device address of the scratch array and the SM count
    struct Dev { bool ready = false; unsigned int* scratch = nullptr; int sms = 0; };
    constexpr int kMaxDev = 64;
    static Dev devs[kMaxDev];
    static std::mutex mu;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDev) return fail(nullptr, GDN_ERR_UNSUPPORTED, "device ordinal beyond 63");
    unsigned int* scratch = nullptr;
    int sms = 0;
    {
        std::lock_guard<std::mutex> lock(mu);
        Dev& d = devs[dev];
        if (!d.ready) {
            void* ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, g_gates_static_scratch);
            if (e != cudaSuccess || !ptr) { cudaGetLastError(); return cuda_fail(nullptr, e, "cudaGetSymbolAddress(static gate scratch)"); }
            e = cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(nullptr, e, "cudaDeviceGetAttribute"); }
            d.scratch = static_cast<unsigned int*>(ptr);
            d.ready = true;
        }
        scratch = d.scratch;
        sms = d.sms;
    }
    // token splits per frame: the rule of gdn_compute_gates (enough CTAs to fill the GPU, at least 64 tokens each), then
    // as many as the scratch holds
    int nspl = (int)((4LL * (sms > 0 ? sms : 148) + BH * F - 1) / (BH * F));
    const int max_spl = (group + 63) / 64;
    if (nspl > max_spl) nspl = max_spl;
    while (nspl > 1 && BH * F * nspl > kStaticGateMaxParts) --nspl;
    if (nspl < 1) nspl = 1;

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // The array keeps what the last call left.  The partial sums are all rewritten before they are read; the counters must
    // start at zero (a call normally leaves them so, but a failed launch would not): cleared in stream order.
    e = cudaMemsetAsync(scratch + kStaticGateMaxParts, 0, (size_t)(BH * F) * sizeof(unsigned int), st);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(nullptr, e, "clearing the static gate counters"); }
    gdn::GateParams gp{};
    gp.x = static_cast<const __nv_bfloat16*>(a->x);
    gp.w_alpha = a->w_alpha; gp.b_alpha = a->b_alpha; gp.a_log = a->a_log; gp.w_beta = a->w_beta; gp.b_beta = a->b_beta;
    gp.alpha_out = alpha_out; gp.beta_out = beta_out;
    gp.part = reinterpret_cast<float*>(scratch);
    gp.counters = scratch + kStaticGateMaxParts;
    gp.x_ts = a->x_token_stride ? a->x_token_stride : (long long)H * D;
    gp.B = B; gp.T = T; gp.H = H; gp.D = D; gp.G = group; gp.F = (int)F; gp.NSPL = nspl;
    gp.log_alpha = log_alpha ? 1 : 0;
    gdn_gates_static_kernel<<<(unsigned int)(BH * F * nspl), gdn::fe::kFeThreads, 0, st>>>(gp);
    e = cudaGetLastError();
    return e == cudaSuccess ? GDN_OK : cuda_fail(nullptr, e, "gdn_gates_static_kernel launch");
}

gdn_status_t gdn_forward_chunk_full(gdn_plan_t* plan, const gdn_featmap_args_t* fm, const void* v, const gdn_gate_args_t* gates,
                                    const float* alpha, const float* beta, const void* out_gate, const float* S_in, const float* z_in,
                                    void* out, float* S_out, float* z_out, gdn_stream_t stream) {
    if (!plan) return fail(nullptr, GDN_ERR_INVALID_ARG, "plan is NULL");
    const gdn_config_t& c = plan->cfg;
    if (!(c.flags & GDN_FLAG_NORMALIZER) || plan->path != GDN_PATH_TC_FRAME)
        return fail(plan, GDN_ERR_UNSUPPORTED, "gdn_forward_chunk_full needs a frame-wise bf16 tensor-core plan created with GDN_FLAG_NORMALIZER");
    gdn_status_t s = fe_check(plan);
    if (s != GDN_OK) return s;
    if (!S_out || !z_out || !out || !v) return fail(plan, GDN_ERR_INVALID_ARG, "a required tensor pointer is NULL");
    if (out_gate && !aligned16(out_gate)) return fail(plan, GDN_ERR_ALIGNMENT, "out_gate must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (c.B == 0 || c.H == 0 || c.T == 0)
        return forward_impl(plan, nullptr, nullptr, nullptr, nullptr, nullptr, alpha, beta, S_in, z_in, out, S_out, z_out, st, true);
    const size_t feat = (size_t)c.B * c.T * c.H * c.d_k;
    if (!plan->fe_feat) {
        if (cudaMalloc(&plan->fe_feat, 4 * feat * 2) != cudaSuccess) { cudaGetLastError(); return fail(plan, GDN_ERR_NOMEM, "feature buffer allocation failed"); }
    }
    __nv_bfloat16* fb = static_cast<__nv_bfloat16*>(plan->fe_feat);
    gdn::FeatmapParams fmp;
    gdn::GateParams gtp;
    bool fm_on = false, g_on = false;
    if (gates) {
        s = fe_gate_buffers(plan);
        if (s != GDN_OK) return s;
        float* a_buf = plan->fe_gates;
        float* b_buf = plan->fe_gates + fe_up4((size_t)c.B * c.H * (c.T / c.group));
        s = gates_fill(plan, gates, a_buf, b_buf, gtp, g_on);
        if (s != GDN_OK) return s;
        alpha = a_buf; beta = b_buf;
    }
    s = featmap_fill(plan, fm, fb, fb + feat, fb + 2 * feat, fb + 3 * feat, fmp, fm_on);
    if (s != GDN_OK) return s;
    auto issue = [&]() {
        gdn_status_t r = launch_frontend(plan, fm_on ? &fmp : nullptr, g_on ? &gtp : nullptr, st, false);
        if (r != GDN_OK) return r;
        return forward_impl(plan, fb, fb + feat, v, fb + 2 * feat, fb + 3 * feat, alpha, beta, S_in, z_in, out, S_out, z_out, st, true,
                            out_gate, true);
    };
    std::vector<const void*> key = {(const void*)3, fm->q, fm->k, fm->rms_wq, fm->rms_wk, fm->rope_cos, fm->rope_sin, v, alpha, beta, out_gate,
                                    S_in, z_in, out, S_out, z_out};
    key.push_back(reinterpret_cast<const void*>((uintptr_t)__float_as_uint_host(fm->rms_eps)));
    if (gates) for (const void* g : {gates->x, (const void*)gates->w_alpha, (const void*)gates->b_alpha, (const void*)gates->a_log,
                                     (const void*)gates->w_beta, (const void*)gates->b_beta, reinterpret_cast<const void*>((uintptr_t)gates->x_token_stride)})
        key.push_back(g);
    return run_graphed(plan, std::move(key), st, issue);
}

gdn_status_t gdn_forward_chunk_host(gdn_plan_t* plan, const void* q_host, const void* k_host, const void* v_host,
                                    const float* alpha_host, const float* beta_host, const float* state_in_host,
                                    void* out_host, float* state_out_host, gdn_stream_t stream) {
    if (!plan) return fail(nullptr, GDN_ERR_INVALID_ARG, "plan is NULL");
    gdn_plan_t* p = plan;
    const gdn_config_t& c = p->cfg;
    if (c.flags & GDN_FLAG_NORMALIZER) return fail(p, GDN_ERR_UNSUPPORTED, "host entry point has no normaliser variant");
    if (c.q_token_stride || c.k_token_stride || c.v_token_stride || c.o_token_stride)
        return fail(p, GDN_ERR_UNSUPPORTED, "host entry point needs dense layouts (token strides 0)");
    if (c.B == 0 || c.H == 0) return GDN_OK;
    if (!state_out_host) return fail(p, GDN_ERR_INVALID_ARG, "state_out_host is NULL");
    if (c.T > 0 && (!q_host || !k_host || !v_host || !alpha_host || !beta_host || !out_host))
        return fail(p, GDN_ERR_INVALID_ARG, "a required host pointer is NULL");
    gdn_status_t ds = check_device(p);
    if (ds != GDN_OK) return ds;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t es = esize(c.io_dtype);
    const size_t nq = (size_t)c.B * c.T * c.H * c.d_k * es, nv = (size_t)c.B * c.T * c.H * c.d_v * es;
    const size_t na = (size_t)c.B * c.H * (c.T / c.group) * 4, nb = (size_t)c.B * c.H * c.T * 4;
    const size_t ns = (size_t)c.B * c.H * c.d_k * c.d_v * 4;
    Staging& h = p->host;
    if (!h.ready) {
        // segmentation: about 16 MB of input per segment (below that the per-copy overheads outweigh the overlap),
        // whole 128-token tiles (G = 1) or whole frames
        const int unit = c.group == 1 ? 128 : c.group;
        const int units = (c.T + unit - 1) / unit;
        int nseg = (int)((2 * nq + nv + na + nb) / (16u << 20));
        // the reverse scan of Alg. 1 l.14-17 runs over ALL frames of the call: a token split is only exact for the forward scan
        if (c.flags & GDN_FLAG_BIDIR) nseg = 1;
        if (nseg > kMaxSeg) nseg = kMaxSeg;
        if (nseg > units) nseg = units;
        if (nseg < 1) nseg = 1;
        h.Tseg = c.T > 0 ? ((units + nseg - 1) / nseg) * unit : 0;
        h.nseg = c.T > 0 ? (c.T + h.Tseg - 1) / h.Tseg : 1;
        h.Ttail = c.T > 0 ? c.T - (h.nseg - 1) * h.Tseg : 0;
        if (h.nseg == 1) { h.Tseg = h.Ttail = c.T; }
        cudaError_t e = cudaSuccess;
        auto alloc = [&](void** ptr, size_t n) { if (e == cudaSuccess) e = cudaMalloc(ptr, n ? n : 16); };
        alloc(&h.q, nq); alloc(&h.k, nq); alloc(&h.v, nv); alloc(&h.out, nv);
        alloc((void**)&h.alpha, na + 16 * kMaxSeg); alloc((void**)&h.beta, nb + 16 * kMaxSeg); alloc((void**)&h.state, ns);
        if (e != cudaSuccess) { cudaGetLastError(); staging_free(h); return fail(p, GDN_ERR_NOMEM, "host-path staging allocation failed"); }
        if (h.nseg > 1) {
            gdn_config_t sc = c;
            sc.T = h.Tseg;
            if (gdn_plan(&sc, &h.seg_plan) != GDN_OK) { staging_free(h); return fail(p, GDN_ERR_NOMEM, std::string("segment plan: ") + g_plan_error); }
            if (h.Ttail != h.Tseg) {
                sc.T = h.Ttail;
                if (gdn_plan(&sc, &h.tail_plan) != GDN_OK) { staging_free(h); return fail(p, GDN_ERR_NOMEM, std::string("tail segment plan: ") + g_plan_error); }
            }
        } else {
            alloc(&h.q2, nq); alloc(&h.k2, nq); alloc(&h.v2, nv);
            alloc((void**)&h.alpha2, na + 16); alloc((void**)&h.beta2, nb + 16);
            if (e != cudaSuccess) { cudaGetLastError(); staging_free(h); return fail(p, GDN_ERR_NOMEM, "host-path staging allocation failed"); }
        }
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h.s_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h.s_out, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h.ev_start, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h.ev_out, cudaEventDisableTiming);
        for (int i = 0; i < (h.nseg > 2 ? h.nseg : 2) && e == cudaSuccess; ++i) {
            e = cudaEventCreateWithFlags(&h.ev_in[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h.ev_comp[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { staging_free(h); return cuda_fail(p, e, "host-path pipeline set-up"); }
        h.ready = true;
        p->workspace_bytes += 2 * nq + 2 * nv + na + nb + ns + (h.nseg == 1 ? 2 * nq + nv + na + nb : 0);
    }
    cudaError_t e = cudaSuccess;
    if (h.nseg == 1) {
        // Small call: one copy in, one launch sequence, one copy out -- pipelined ACROSS calls.  q, k, v, alpha, beta go to the
        // staging set of this call's parity on the internal copy-in stream; that stream waits only for the compute that last
        // read the set (two calls ago), NOT for the work queued on `st`: host inputs hold their data when the call is made
        // (include/gdn.h), so the copy-in of call i+1 runs while call i computes and copies out.  Exceptions, in stream order as
        // before: state_in_host (a stream of chunks hands the state through host memory), and every input when it overlaps a
        // host buffer the previous call writes.
        const int par = (int)(h.calls & 1ull);
        void *dq = par ? h.q2 : h.q, *dk = par ? h.k2 : h.k, *dv = par ? h.v2 : h.v;
        float *da = par ? h.alpha2 : h.alpha, *db = par ? h.beta2 : h.beta;
        auto ck1 = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
        auto overlaps_prev = [&](const void* ptr, size_t n) {
            const char* lo = static_cast<const char*>(ptr);
            for (int i = 0; i < 2; ++i)
                if (h.prev_out_lo[i] && lo < static_cast<const char*>(h.prev_out_hi[i]) && lo + n > static_cast<const char*>(h.prev_out_lo[i])) return true;
            return false;
        };
        const bool chained = overlaps_prev(q_host, nq) || overlaps_prev(k_host, nq) || overlaps_prev(v_host, nv) ||
                             overlaps_prev(alpha_host, na) || overlaps_prev(beta_host, nb);
        // (two copy-in streams: one host->device copy stream alone reaches 37-48 GB/s on this class of host, two fill the link)
        if (chained || h.calls == 0) {
            ck1(cudaEventRecord(h.ev_start, st));
            ck1(cudaStreamWaitEvent(h.s_in, h.ev_start, 0));
            ck1(cudaStreamWaitEvent(h.s_out, h.ev_start, 0));
        }
        if (h.calls >= 2) {                            // the set's last reader is done
            ck1(cudaStreamWaitEvent(h.s_in, h.ev_comp[par], 0));
            ck1(cudaStreamWaitEvent(h.s_out, h.ev_comp[par], 0));
        }
        auto h2d = [&](void* d, const void* s, size_t n, cudaStream_t cs) { if (e == cudaSuccess && n) e = cudaMemcpyAsync(d, s, n, cudaMemcpyHostToDevice, cs); };
        h2d(dq, q_host, nq, h.s_in); h2d(da, alpha_host, na, h.s_in); h2d(db, beta_host, nb, h.s_in);
        h2d(dk, k_host, nq / 2, h.s_in);
        h2d(static_cast<char*>(dk) + nq / 2, static_cast<const char*>(k_host) + nq / 2, nq - nq / 2, h.s_out);
        h2d(dv, v_host, nv, h.s_out);
        ck1(cudaEventRecord(h.ev_in[par], h.s_in));
        ck1(cudaEventRecord(h.ev_out, h.s_out));
        if (state_in_host) h2d(h.state, state_in_host, ns, st);
        ck1(cudaStreamWaitEvent(st, h.ev_in[par], 0));
        ck1(cudaStreamWaitEvent(st, h.ev_out, 0));
        if (e != cudaSuccess) return cuda_fail(p, e, "host->device copy");
        gdn_status_t fs = forward_impl(p, dq, dk, dv, nullptr, nullptr, da, db,
                                       state_in_host ? h.state : nullptr, nullptr, h.out, h.state, nullptr, st, false);
        if (fs != GDN_OK) return fs;
        ck1(cudaEventRecord(h.ev_comp[par], st));
        if (nv) ck1(cudaMemcpyAsync(out_host, h.out, nv, cudaMemcpyDeviceToHost, st));
        ck1(cudaMemcpyAsync(state_out_host, h.state, ns, cudaMemcpyDeviceToHost, st));
        if (e != cudaSuccess) return cuda_fail(p, e, "device->host copy");
        h.prev_out_lo[0] = out_host; h.prev_out_hi[0] = static_cast<const char*>(out_host) + nv;
        h.prev_out_lo[1] = state_out_host; h.prev_out_hi[1] = reinterpret_cast<const char*>(state_out_host) + ns;
        ++h.calls;
        return GDN_OK;
    }
    // ---- pipelined: copy-in stream | caller's stream (compute) | copy-out stream --------------------------------
    auto ck = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    ck(cudaEventRecord(h.ev_start, st));               // everything queued on `st` before this call comes first
    ck(cudaStreamWaitEvent(h.s_in, h.ev_start, 0));
    ck(cudaStreamWaitEvent(h.s_out, h.ev_start, 0));
    if (state_in_host) ck(cudaMemcpyAsync(h.state, state_in_host, ns, cudaMemcpyHostToDevice, h.s_in));
    const size_t rowq = (size_t)c.H * c.d_k * es, rowv = (size_t)c.H * c.d_v * es;      // bytes per token
    const int BH = c.B * c.H;
    size_t oq = 0, ov = 0, oa = 0, ob = 0;              // byte offsets of the segment inside the staging buffers
    for (int sgi = 0; sgi < h.nseg; ++sgi) {
        const int t0 = sgi * h.Tseg, Ts = (sgi == h.nseg - 1) ? h.Ttail : h.Tseg;
        const int Fs = Ts / c.group, f0 = t0 / c.group, Ftot = c.T / c.group;
        uint8_t *dq = (uint8_t*)h.q + oq, *dk = (uint8_t*)h.k + oq, *dv = (uint8_t*)h.v + ov, *dout = (uint8_t*)h.out + ov;
        float *da = (float*)((uint8_t*)h.alpha + oa), *db = (float*)((uint8_t*)h.beta + ob);
        // [B,T,H,d] -> compact [B,Ts,H,d]: B rows of Ts*H*d elements, source pitch T*H*d
        ck(cudaMemcpy2DAsync(dq, Ts * rowq, (const uint8_t*)q_host + t0 * rowq, c.T * rowq, Ts * rowq, c.B, cudaMemcpyHostToDevice, h.s_in));
        ck(cudaMemcpy2DAsync(dk, Ts * rowq, (const uint8_t*)k_host + t0 * rowq, c.T * rowq, Ts * rowq, c.B, cudaMemcpyHostToDevice, h.s_in));
        ck(cudaMemcpy2DAsync(dv, Ts * rowv, (const uint8_t*)v_host + t0 * rowv, c.T * rowv, Ts * rowv, c.B, cudaMemcpyHostToDevice, h.s_in));
        // [B,H,T/G] -> [B,H,Ts/G] and [B,H,T] -> [B,H,Ts]
        ck(cudaMemcpy2DAsync(da, (size_t)Fs * 4, alpha_host + f0, (size_t)Ftot * 4, (size_t)Fs * 4, BH, cudaMemcpyHostToDevice, h.s_in));
        ck(cudaMemcpy2DAsync(db, (size_t)Ts * 4, beta_host + t0, (size_t)c.T * 4, (size_t)Ts * 4, BH, cudaMemcpyHostToDevice, h.s_in));
        ck(cudaEventRecord(h.ev_in[sgi], h.s_in));
        if (e != cudaSuccess) return cuda_fail(p, e, "host->device segment copy");
        ck(cudaStreamWaitEvent(st, h.ev_in[sgi], 0));
        gdn_plan_t* sp = (Ts == h.Tseg) ? h.seg_plan : h.tail_plan;
        const float* sin = (sgi == 0 && !state_in_host) ? nullptr : h.state;
        gdn_status_t fs = forward_impl(sp, dq, dk, dv, nullptr, nullptr, da, db, sin, nullptr, dout, h.state, nullptr, st, false);
        if (fs != GDN_OK) return fail(p, fs, std::string("segment forward: ") + sp->err);
        ck(cudaEventRecord(h.ev_comp[sgi], st));
        ck(cudaStreamWaitEvent(h.s_out, h.ev_comp[sgi], 0));
        ck(cudaMemcpy2DAsync((uint8_t*)out_host + t0 * rowv, c.T * rowv, dout, Ts * rowv, Ts * rowv, c.B, cudaMemcpyDeviceToHost, h.s_out));
        oq += (size_t)c.B * Ts * rowq; ov += (size_t)c.B * Ts * rowv;
        oa = (oa + (size_t)BH * Fs * 4 + 15) & ~(size_t)15;     // every segment's gates start 16-byte aligned (forward_impl checks it)
        ob = (ob + (size_t)BH * Ts * 4 + 15) & ~(size_t)15;
    }
    ck(cudaMemcpyAsync(state_out_host, h.state, ns, cudaMemcpyDeviceToHost, st));
    ck(cudaEventRecord(h.ev_out, h.s_out));
    ck(cudaStreamWaitEvent(st, h.ev_out, 0));          // `stream` completes only when every output byte is on the host
    if (e != cudaSuccess) return cuda_fail(p, e, "host pipeline");
    return GDN_OK;
}

gdn_status_t gdn_destroy(gdn_plan_t* plan) {
    if (plan) { for (auto& g : plan->graphs) if (g.exec) cudaGraphExecDestroy(g.exec); plan->graphs.clear(); }
    if (plan) { if (plan->fe_feat) cudaFree(plan->fe_feat); if (plan->fe_gates) cudaFree(plan->fe_gates); plan->fe_feat = nullptr; plan->fe_gates = nullptr; }
    if (!plan) return GDN_OK;
    gdn::tc_plan_free(plan->tc);
    plan->prof.set_enabled(false);
    if (plan->z_stage) cudaFree(plan->z_stage);
    staging_free(plan->host);
    delete plan;
    return GDN_OK;
}

gdn_status_t gdn_plan_get_info(const gdn_plan_t* plan, gdn_plan_info_t* info) {
    if (!plan || !info) return GDN_ERR_INVALID_ARG;
    info->path = plan->path;
    info->chunk = plan->chunk;
    info->launches_per_call = plan->launches;
    info->sm_count = plan->sm_count;
    info->workspace_bytes = plan->workspace_bytes;
    return GDN_OK;
}

gdn_status_t gdn_plan_set_profiling(gdn_plan_t* plan, int enable) {
    if (!plan) return GDN_ERR_INVALID_ARG;
    plan->prof.set_enabled(enable != 0);
    return GDN_OK;
}

gdn_status_t gdn_plan_kernel_times(gdn_plan_t* plan, int max_n, const char** names, float* avg_ms, int* n_out) {
    if (!plan || !names || !avg_ms || !n_out || max_n < 0) return GDN_ERR_INVALID_ARG;
    *n_out = plan->prof.collect(max_n, names, avg_ms);
    return GDN_OK;
}

const char* gdn_status_string(gdn_status_t s) {
    switch (s) {
        case GDN_OK: return "GDN_OK";
        case GDN_ERR_INVALID_ARG: return "GDN_ERR_INVALID_ARG";
        case GDN_ERR_UNSUPPORTED: return "GDN_ERR_UNSUPPORTED";
        case GDN_ERR_ALIGNMENT: return "GDN_ERR_ALIGNMENT";
        case GDN_ERR_NOMEM: return "GDN_ERR_NOMEM";
        case GDN_ERR_ARCH: return "GDN_ERR_ARCH";
        case GDN_ERR_CUDA: return "GDN_ERR_CUDA";
    }
    return "GDN_ERR_UNKNOWN";
}

const char* gdn_last_error(const gdn_plan_t* plan) { return plan ? plan->err.c_str() : g_plan_error.c_str(); }

const char* gdn_version(void) { return "0.1.0"; }

}  // extern "C"
