// ann_static.cu -- df_chem_ann_source_static: the tensor-path ANN source term (H3) for callers that may not allocate
// device memory and have no workspace to hand in (code under stream capture, serving loops, harnesses that forbid
// cudaMalloc).  Same kernel as df_chem_ann_source (ann_bf16.cu), same results; the per-CTA H2 scratch of that kernel lives
// in a file-scope __device__ array of this translation unit instead of a caller-supplied workspace.
//
// Cost and limits (also in include/df_thermo.h):
//   * every GPU that loads libdfthermo.so holds DF_ANN_STATIC_SCRATCH_BYTES (32 MiB) of device memory until the process
//     exits, whether or not this entry point is ever called;
//   * a call whose scratch need, df_ann_workspace_bytes(ann, n_cells), exceeds that is rejected (DF_ERR_UNSUPPORTED): the
//     need is min(ceil(n_cells/128), SMs) x ceil(d2/64) x 16 KB, e.g. 148 x 13 x 16 KB = 29.4 MiB for the
//     21-1600-800-400-19 network at any n_cells on a 148-SM part;
//   * all calls on a device share the one array: two calls that overlap on the GPU (different streams, no dependency
//     between them) race on it.  Calls on one stream, or ordered by events, are safe: every tile writes its H2 chunks
//     before it reads them, so nothing has to start at zero and nothing is carried from one call to the next.
#include <mutex>

#include "ann_common.cuh"

namespace {

constexpr size_t kStaticScratchBytes = (size_t)DF_ANN_STATIC_SCRATCH_BYTES;
constexpr int kMaxDevices = 128;

// In host code this name is only a handle for the runtime's symbol table -- never a device address: the address is
// looked up with cudaGetSymbolAddress, per device, with that device current (each device has its own copy).
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

std::mutex g_addr_mutex;
void* g_scratch_addr[kMaxDevices] = {};   // device address of g_static_scratch on device i, once looked up

df_status static_scratch(void** out) {
    int dev = -1;
    DF_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices)
        return df_set_error(DF_ERR_UNSUPPORTED, "df_chem_ann_source_static: device ordinal %d not supported (max %d)", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_addr_mutex);
    if (!g_scratch_addr[dev]) {
        void* ptr = nullptr;
        DF_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_scratch));
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u))
            return df_set_error(DF_ERR_CUDA, "df_chem_ann_source_static: bad address for the static scratch on device %d", dev);
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return DF_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

extern "C" size_t df_ann_static_scratch_bytes(void) { return kStaticScratchBytes; }

extern "C" df_status df_chem_ann_source_static(const df_ann* ann, const df_mech* mech, long long n, long long ld,
                                               const float* T, const float* p, const float* Y, float* omega, float* dY,
                                               void* stream) {
    const char* fn = "df_chem_ann_source_static";
    if (!ann || !mech) return df_set_error(DF_ERR_INVALID_ARG, "%s: NULL handle", fn);
    if (ann->K != mech->K) return df_set_error(DF_ERR_INVALID_ARG, "%s: ann has K=%d, mech has K=%d", fn, ann->K, mech->K);
    if (ann->precision != 1 || !ann->bf16)
        return df_set_error(DF_ERR_UNSUPPORTED, "%s: the handle is not on the tensor path (precision 1); the fp32 path needs no "
                            "workspace -- call df_chem_ann_source with workspace = NULL", fn);
    if (n < 0 || ld < n || ld % 4 != 0) return df_set_error(DF_ERR_INVALID_ARG, "%s: bad n_cells / ld", fn);
    // the per-device set-up (symbol lookup) also runs for n_cells == 0, so that a caller can do it ahead of a capture
    void* scratch = nullptr;
    const df_status st = static_scratch(&scratch);
    if (st != DF_OK) return st;
    if (n == 0) return DF_OK;
    if (!T || !p || !Y) return df_set_error(DF_ERR_INVALID_ARG, "%s: NULL input field", fn);
    if (!omega && !dY) return DF_OK;
    if (!aligned16(T) || !aligned16(p) || !aligned16(Y) || !aligned16(omega) || !aligned16(dY))
        return df_set_error(DF_ERR_INVALID_ARG, "%s: fields must be 16-byte aligned", fn);
    const size_t need = ann_bf16_workspace(ann, n);
    if (need > kStaticScratchBytes)
        return df_set_error(DF_ERR_UNSUPPORTED, "%s: this network and n_cells need %zu bytes of scratch, the static scratch holds %zu; "
                            "use df_chem_ann_source with a workspace", fn, need, kStaticScratchBytes);
    return launch_ann_bf16(ann, mech, n, ld, T, p, Y, omega, dY, scratch, kStaticScratchBytes, (cudaStream_t)stream);
}
