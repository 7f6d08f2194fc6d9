// api.cu -- the extern "C" boundary of libdfthermo.so (include/df_thermo.h): argument validation,
// df_ann create/destroy, dispatch to the kernel launchers, and the host-buffer step used by
// bench.py's e2e leg.  No CPU fallback anywhere: every path ends in a kernel launch or an error.
#include <cmath>
#include <cstring>
#include <new>

#include "common.cuh"

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

df_status check_fields(const char* fn, long long n, long long ld) {
    if (n < 0) return df_set_error(DF_ERR_INVALID_ARG, "%s: n_cells < 0", fn);
    if (ld < n) return df_set_error(DF_ERR_INVALID_ARG, "%s: ld (%lld) < n_cells (%lld)", fn, ld, n);
    if (ld % 4 != 0) return df_set_error(DF_ERR_INVALID_ARG, "%s: ld (%lld) must be a multiple of 4", fn, ld);
    return DF_OK;
}

}  // namespace

extern "C" df_status df_ann_create(df_ann** out, int n_layers, const int* dims, const float* const* W,
                                   const float* const* b, int precision, const double* x_mean, const double* x_std,
                                   const double* u_mean, const double* u_std, double boxcox_lambda, double dt) {
    if (!out) return df_set_error(DF_ERR_INVALID_ARG, "df_ann_create: out is NULL");
    *out = nullptr;
    if (!dims || !W || !b || !x_mean || !x_std || !u_mean || !u_std)
        return df_set_error(DF_ERR_INVALID_ARG, "df_ann_create: NULL argument");
    if (n_layers < 1 || n_layers > 8) return df_set_error(DF_ERR_UNSUPPORTED, "df_ann_create: n_layers=%d", n_layers);
    if (precision != 0 && precision != 1) return df_set_error(DF_ERR_INVALID_ARG, "df_ann_create: precision=%d", precision);
    const int K = dims[n_layers];
    if (K < 1 || K > DF_MAX_K || dims[0] != K + 2)
        return df_set_error(DF_ERR_INVALID_ARG, "df_ann_create: need dims[0] == dims[n_layers] + 2, K in [1,%d]", DF_MAX_K);
    if (!(boxcox_lambda > 0.0) || !(dt > 0.0))
        return df_set_error(DF_ERR_INVALID_ARG, "df_ann_create: boxcox_lambda and dt must be > 0");
    for (int l = 0; l < n_layers; ++l)
        if (!W[l] || !b[l] || dims[l + 1] < 1) return df_set_error(DF_ERR_INVALID_ARG, "df_ann_create: layer %d", l);
    for (int i = 0; i < K + 2; ++i)
        if (!(x_std[i] > 0.0)) return df_set_error(DF_ERR_INVALID_ARG, "df_ann_create: x_std[%d] <= 0", i);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return df_set_error(DF_ERR_CUDA, "df_ann_create: no CUDA device (there is no CPU fallback)");

    df_ann* a = new (std::nothrow) df_ann;
    if (!a) return df_set_error(DF_ERR_ALLOC, "df_ann_create: out of host memory");
    a->n_layers = n_layers;
    a->dims.assign(dims, dims + n_layers + 1);
    a->precision = precision;
    a->K = K;
    memset(&a->norm, 0, sizeof(a->norm));
    for (int i = 0; i < K + 2; ++i) {
        a->norm.x_mean[i] = (float)x_mean[i];
        a->norm.x_inv_std[i] = (float)(1.0 / x_std[i]);
    }
    for (int k = 0; k < K; ++k) {
        a->norm.u_mean[k] = (float)u_mean[k];
        a->norm.u_std[k] = (float)u_std[k];
    }
    a->norm.lambda = (float)boxcox_lambda;
    a->norm.inv_lambda = (float)(1.0 / boxcox_lambda);
    a->norm.inv_dt = (float)(1.0 / dt);

    if (precision == 0) {
        for (int l = 0; l <= n_layers; ++l)
            if (dims[l] > 256) {
                delete a;
                return df_set_error(DF_ERR_UNSUPPORTED, "df_ann_create: fp32 path supports layer widths <= 256 (got %d)", dims[l]);
            }
        std::vector<float> host;
        for (int l = 0; l < n_layers; ++l) {
            const int din = dims[l], dout = dims[l + 1], op = (dout + 7) / 8 * 8;
            a->out_pad.push_back(op);
            a->w32_off.push_back(host.size());
            host.resize(host.size() + (size_t)din * op, 0.f);
            float* wt = host.data() + a->w32_off[l];
            for (int o = 0; o < dout; ++o)
                for (int i = 0; i < din; ++i) wt[(size_t)i * op + o] = W[l][(size_t)o * din + i];
            a->b32_off.push_back(host.size());
            host.resize(host.size() + op, 0.f);
            memcpy(host.data() + a->b32_off[l], b[l], sizeof(float) * dout);
        }
        if (cudaMalloc((void**)&a->w32, host.size() * sizeof(float)) != cudaSuccess) {
            delete a;
            return df_set_error(DF_ERR_ALLOC, "df_ann_create: cudaMalloc failed");
        }
        if (cudaMemcpy(a->w32, host.data(), host.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) {
            df_ann_destroy(a);
            return df_set_error(DF_ERR_CUDA, "df_ann_create: cudaMemcpy failed");
        }
    } else {
        const df_status st = ann_bf16_create(a, W, b);
        if (st != DF_OK) {
            df_ann_destroy(a);
            return st;
        }
    }
    *out = a;
    return DF_OK;
}

extern "C" df_status df_ann_destroy(df_ann* ann) {
    if (!ann) return DF_OK;
    cudaFree(ann->w32);
    if (ann->bf16) ann_bf16_destroy(ann);
    delete ann;
    return DF_OK;
}

extern "C" size_t df_ann_workspace_bytes(const df_ann* ann, long long n_cells) {
    if (!ann || n_cells <= 0 || ann->precision == 0) return 0;
    return ann_bf16_workspace(ann, n_cells);
}

extern "C" df_status df_thermo_T_from_h(const df_mech* mech, long long n, long long ld, const float* h,
                                        const float* Y, float* T, float* cp, int* n_unconverged, void* stream) {
    if (!mech) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_T_from_h: mech is NULL");
    df_status st = check_fields("df_thermo_T_from_h", n, ld);
    if (st != DF_OK) return st;
    if (n == 0) return DF_OK;
    if (!h || !Y || !T) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_T_from_h: NULL field");
    if (!aligned16(h) || !aligned16(Y) || !aligned16(T) || !aligned16(cp))
        return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_T_from_h: fields must be 16-byte aligned");
    return launch_T_from_h(mech, n, ld, h, Y, T, cp, n_unconverged, (cudaStream_t)stream);
}

extern "C" df_status df_thermo_properties(const df_mech* mech, long long n, long long ld, const float* T,
                                          const float* p, const float* Y, float* cp, float* h, float* mu,
                                          float* lambda, float* D, void* stream) {
    if (!mech) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_properties: mech is NULL");
    df_status st = check_fields("df_thermo_properties", n, ld);
    if (st != DF_OK) return st;
    if (n == 0) return DF_OK;
    if (!T || !Y || (D && !p)) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_properties: NULL input field");
    if (!cp && !h && !mu && !lambda && !D) return DF_OK;
    if (!aligned16(T) || !aligned16(p) || !aligned16(Y) || !aligned16(cp) || !aligned16(h) || !aligned16(mu) ||
        !aligned16(lambda) || !aligned16(D))
        return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_properties: fields must be 16-byte aligned");
    return launch_properties(mech, n, ld, T, p, Y, cp, h, mu, lambda, D, (cudaStream_t)stream);
}

extern "C" df_status df_chem_ann_source(const df_ann* ann, const df_mech* mech, long long n, long long ld,
                                        const float* T, const float* p, const float* Y, float* omega, float* dY,
                                        void* workspace, size_t workspace_bytes, void* stream) {
    if (!ann || !mech) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source: NULL handle");
    if (ann->K != mech->K)
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source: ann has K=%d, mech has K=%d", ann->K, mech->K);
    df_status st = check_fields("df_chem_ann_source", n, ld);
    if (st != DF_OK) return st;
    if (n == 0) return DF_OK;
    if (!T || !p || !Y) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source: NULL input field");
    if (!omega && !dY) return DF_OK;
    if (!aligned16(T) || !aligned16(p) || !aligned16(Y) || !aligned16(omega) || !aligned16(dY))
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source: fields must be 16-byte aligned");
    if (ann->precision == 0) return launch_ann_fp32(ann, mech, n, ld, T, p, Y, omega, dY, (cudaStream_t)stream);
    const size_t need = ann_bf16_workspace(ann, n);
    if (need > 0 && (!workspace || workspace_bytes < need))
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source: workspace of %zu bytes needed, %zu given", need,
                            workspace ? workspace_bytes : (size_t)0);
    if (reinterpret_cast<uintptr_t>(workspace) & 1023u)
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source: workspace must be 1024-byte aligned");
    return launch_ann_bf16(ann, mech, n, ld, T, p, Y, omega, dY, workspace, workspace_bytes, (cudaStream_t)stream);
}

// ---- host-buffer step ----------------------------------------------------------------------------
// df_step_host pipelines the step over up to kHostChunks slices of the cells: copy-in of slice c+1 and copy-out of
// slice c-1 overlap the kernels of slice c (PCIe is full duplex, cells are independent).
constexpr int kHostChunks = 8;
constexpr long long kHostChunkMin = 65536;   // cells; below this a slice no longer fills the GPU

struct df_host_ctx {
    const df_mech* mech;
    const df_ann* ann;
    long long cap;  // cells (pitch of the staging arrays)
    cudaStream_t stream;             // compute
    cudaStream_t s_in, s_out;        // host->device and device->host copies (one copy engine each)
    cudaEvent_t ev_in[kHostChunks], ev_done[kHostChunks], ev_prev;
    float *h, *p, *T, *Y, *cp, *mu, *lam, *D, *omega;
    void* ws;
    size_t ws_bytes;
};

extern "C" df_status df_host_ctx_create(df_host_ctx** out, const df_mech* mech, const df_ann* ann, long long max_cells) {
    if (!out || !mech || max_cells < 1) return df_set_error(DF_ERR_INVALID_ARG, "df_host_ctx_create: bad argument");
    *out = nullptr;
    if (ann && ann->K != mech->K) return df_set_error(DF_ERR_INVALID_ARG, "df_host_ctx_create: K mismatch");
    df_host_ctx* c = new (std::nothrow) df_host_ctx;
    if (!c) return df_set_error(DF_ERR_ALLOC, "df_host_ctx_create: out of host memory");
    memset(c, 0, sizeof(*c));
    c->mech = mech;
    c->ann = ann;
    c->cap = (max_cells + 255) / 256 * 256;
    const size_t f = (size_t)c->cap * sizeof(float), K = (size_t)mech->K;
    c->ws_bytes = ann ? df_ann_workspace_bytes(ann, max_cells) : 0;
    bool ok = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->ev_prev, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; ok && i < kHostChunks; ++i)
        ok = cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&c->h, f) == cudaSuccess && cudaMalloc((void**)&c->p, f) == cudaSuccess &&
         cudaMalloc((void**)&c->T, f) == cudaSuccess && cudaMalloc((void**)&c->Y, f * K) == cudaSuccess &&
         cudaMalloc((void**)&c->cp, f) == cudaSuccess && cudaMalloc((void**)&c->mu, f) == cudaSuccess &&
         cudaMalloc((void**)&c->lam, f) == cudaSuccess && cudaMalloc((void**)&c->D, f * K) == cudaSuccess &&
         cudaMalloc((void**)&c->omega, f * K) == cudaSuccess;
    if (ok && c->ws_bytes) ok = cudaMalloc(&c->ws, c->ws_bytes) == cudaSuccess;
    if (!ok) {
        df_host_ctx_destroy(c);
        return df_set_error(DF_ERR_ALLOC, "df_host_ctx_create: device allocation failed: %s",
                            cudaGetErrorString(cudaGetLastError()));
    }
    *out = c;
    return DF_OK;
}

extern "C" df_status df_host_ctx_destroy(df_host_ctx* c) {
    if (!c) return DF_OK;
    cudaFree(c->h); cudaFree(c->p); cudaFree(c->T); cudaFree(c->Y); cudaFree(c->cp); cudaFree(c->mu);
    cudaFree(c->lam); cudaFree(c->D); cudaFree(c->omega); cudaFree(c->ws);
    for (int i = 0; i < kHostChunks; ++i) {
        if (c->ev_in[i]) cudaEventDestroy(c->ev_in[i]);
        if (c->ev_done[i]) cudaEventDestroy(c->ev_done[i]);
    }
    if (c->ev_prev) cudaEventDestroy(c->ev_prev);
    if (c->stream) cudaStreamDestroy(c->stream);
    if (c->s_in) cudaStreamDestroy(c->s_in);
    if (c->s_out) cudaStreamDestroy(c->s_out);
    delete c;
    return DF_OK;
}

extern "C" df_status df_step_host(df_host_ctx* c, long long n, long long ld, const float* h, const float* p,
                                  const float* T_guess, const float* Y, float* T, float* cp, float* mu, float* lambda,
                                  float* D, float* omega) {
    if (!c) return df_set_error(DF_ERR_INVALID_ARG, "df_step_host: ctx is NULL");
    if (n < 0 || ld < n || n > c->cap) return df_set_error(DF_ERR_INVALID_ARG, "df_step_host: bad n_cells/ld");
    if (n == 0) return DF_OK;
    if (!h || !p || !T_guess || !Y) return df_set_error(DF_ERR_INVALID_ARG, "df_step_host: NULL input");
    if (omega && !c->ann) return df_set_error(DF_ERR_INVALID_ARG, "df_step_host: omega requested but ctx has no ann");
    const int K = c->mech->K;
    const size_t dpitch = (size_t)c->cap * sizeof(float), hpitch = (size_t)ld * sizeof(float);
    // slices of m cells (a multiple of 1024: tile and vector-load alignment of every kernel)
    long long m = (n + kHostChunks - 1) / kHostChunks;
    if (m < kHostChunkMin) m = kHostChunkMin;
    m = (m + 1023) / 1024 * 1024;
    const int nch = (int)((n + m - 1) / m);
    // the staging buffers are reused: this call's copies-in must not overtake the previous call's kernels/copies-out
    // (df_step_host synchronises before it returns, so this only matters after an error return)
    DF_CUDA_TRY(cudaEventRecord(c->ev_prev, c->s_out));
    DF_CUDA_TRY(cudaStreamWaitEvent(c->s_in, c->ev_prev, 0));
    for (int ch = 0; ch < nch; ++ch) {
        const long long o = (long long)ch * m, nc = (n - o < m) ? n - o : m;
        const size_t f = (size_t)nc * sizeof(float);
        DF_CUDA_TRY(cudaMemcpyAsync(c->h + o, h + o, f, cudaMemcpyHostToDevice, c->s_in));
        DF_CUDA_TRY(cudaMemcpyAsync(c->p + o, p + o, f, cudaMemcpyHostToDevice, c->s_in));
        DF_CUDA_TRY(cudaMemcpyAsync(c->T + o, T_guess + o, f, cudaMemcpyHostToDevice, c->s_in));
        DF_CUDA_TRY(cudaMemcpy2DAsync(c->Y + o, dpitch, Y + o, hpitch, f, K, cudaMemcpyHostToDevice, c->s_in));
        DF_CUDA_TRY(cudaEventRecord(c->ev_in[ch], c->s_in));

        DF_CUDA_TRY(cudaStreamWaitEvent(c->stream, c->ev_in[ch], 0));
        df_status st = df_thermo_T_from_h(c->mech, nc, c->cap, c->h + o, c->Y + o, c->T + o, nullptr, nullptr, c->stream);
        if (st != DF_OK) return st;
        st = df_thermo_properties(c->mech, nc, c->cap, c->T + o, c->p + o, c->Y + o, cp ? c->cp + o : nullptr, nullptr,
                                  mu ? c->mu + o : nullptr, lambda ? c->lam + o : nullptr, D ? c->D + o : nullptr, c->stream);
        if (st != DF_OK) return st;
        if (omega) {
            st = df_chem_ann_source(c->ann, c->mech, nc, c->cap, c->T + o, c->p + o, c->Y + o, c->omega + o, nullptr, c->ws,
                                    c->ws_bytes, c->stream);
            if (st != DF_OK) return st;
        }
        DF_CUDA_TRY(cudaEventRecord(c->ev_done[ch], c->stream));

        DF_CUDA_TRY(cudaStreamWaitEvent(c->s_out, c->ev_done[ch], 0));
        if (T) DF_CUDA_TRY(cudaMemcpyAsync(T + o, c->T + o, f, cudaMemcpyDeviceToHost, c->s_out));
        if (cp) DF_CUDA_TRY(cudaMemcpyAsync(cp + o, c->cp + o, f, cudaMemcpyDeviceToHost, c->s_out));
        if (mu) DF_CUDA_TRY(cudaMemcpyAsync(mu + o, c->mu + o, f, cudaMemcpyDeviceToHost, c->s_out));
        if (lambda) DF_CUDA_TRY(cudaMemcpyAsync(lambda + o, c->lam + o, f, cudaMemcpyDeviceToHost, c->s_out));
        if (D) DF_CUDA_TRY(cudaMemcpy2DAsync(D + o, hpitch, c->D + o, dpitch, f, K, cudaMemcpyDeviceToHost, c->s_out));
        if (omega) DF_CUDA_TRY(cudaMemcpy2DAsync(omega + o, hpitch, c->omega + o, dpitch, f, K, cudaMemcpyDeviceToHost, c->s_out));
    }
    DF_CUDA_TRY(cudaStreamSynchronize(c->s_out));
    DF_CUDA_TRY(cudaStreamSynchronize(c->stream));
    return DF_OK;
}

// ---- single-launch step ---------------------------------------------------------------------------
// P:34 "to avoid the CPU-GPU memory copy overhead, the entire computational process is executed on GPU": a solver calls
// the update every time step on the same field arrays, so the whole step -- guess copy, T_from_h, properties, ANN
// source -- is captured once as a CUDA graph and replayed with ONE launch per time step.
struct df_step_plan {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    int n_kernels = 0;
};

extern "C" df_status df_step_plan_destroy(df_step_plan* p) {
    if (!p) return DF_OK;
    if (p->exec) cudaGraphExecDestroy(p->exec);
    if (p->graph) cudaGraphDestroy(p->graph);
    delete p;
    return DF_OK;
}

extern "C" df_status df_step_plan_create(df_step_plan** out, const df_mech* mech, const df_ann* ann, long long n, long long ld,
                                         const float* h, const float* p, const float* T_guess, const float* Y, float* T,
                                         float* cp, float* mu, float* lambda, float* D, float* omega, void* workspace,
                                         size_t workspace_bytes) {
    if (!out) return df_set_error(DF_ERR_INVALID_ARG, "df_step_plan_create: out is NULL");
    *out = nullptr;
    if (!mech || n < 1 || !h || !Y || !T) return df_set_error(DF_ERR_INVALID_ARG, "df_step_plan_create: bad argument");
    if (omega && !ann) return df_set_error(DF_ERR_INVALID_ARG, "df_step_plan_create: omega requested but ann is NULL");
    df_step_plan* pl = new (std::nothrow) df_step_plan;
    if (!pl) return df_set_error(DF_ERR_ALLOC, "df_step_plan_create: out of host memory");
    cudaStream_t cs = nullptr;
    if (cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) != cudaSuccess) {
        delete pl;
        return df_set_error(DF_ERR_CUDA, "df_step_plan_create: cudaStreamCreate failed");
    }
    df_status st = DF_OK;
    cudaError_t ce = cudaStreamBeginCapture(cs, cudaStreamCaptureModeRelaxed);
    if (ce != cudaSuccess) st = df_set_error(DF_ERR_CUDA, "df_step_plan_create: cudaStreamBeginCapture: %s", cudaGetErrorString(ce));
    if (st == DF_OK) {
        if (T_guess && T_guess != T && cudaMemcpyAsync(T, T_guess, (size_t)n * sizeof(float), cudaMemcpyDeviceToDevice, cs) != cudaSuccess)
            st = df_set_error(DF_ERR_CUDA, "df_step_plan_create: guess copy failed");
        if (st == DF_OK) st = df_thermo_T_from_h(mech, n, ld, h, Y, T, nullptr, nullptr, cs);
        if (st == DF_OK) ++pl->n_kernels;
        if (st == DF_OK && (cp || mu || lambda || D)) {
            st = df_thermo_properties(mech, n, ld, T, p, Y, cp, nullptr, mu, lambda, D, cs);
            if (st == DF_OK) ++pl->n_kernels;
        }
        if (st == DF_OK && omega) {
            st = df_chem_ann_source(ann, mech, n, ld, T, p, Y, omega, nullptr, workspace, workspace_bytes, cs);
            if (st == DF_OK) ++pl->n_kernels;
        }
        ce = cudaStreamEndCapture(cs, &pl->graph);   // always ends the capture, also after an error above
        if (st == DF_OK && ce != cudaSuccess) st = df_set_error(DF_ERR_CUDA, "df_step_plan_create: cudaStreamEndCapture: %s", cudaGetErrorString(ce));
    }
    if (st == DF_OK) {
        ce = cudaGraphInstantiate(&pl->exec, pl->graph, 0);
        if (ce != cudaSuccess) st = df_set_error(DF_ERR_CUDA, "df_step_plan_create: cudaGraphInstantiate: %s", cudaGetErrorString(ce));
    }
    cudaStreamDestroy(cs);
    if (st != DF_OK) {
        df_step_plan_destroy(pl);
        return st;
    }
    *out = pl;
    return DF_OK;
}

extern "C" df_status df_thermochem_step(df_step_plan* plan, void* stream) {
    if (!plan || !plan->exec) return df_set_error(DF_ERR_INVALID_ARG, "df_thermochem_step: plan is NULL");
    DF_CUDA_TRY(cudaGraphLaunch(plan->exec, (cudaStream_t)stream));
    return DF_OK;
}
