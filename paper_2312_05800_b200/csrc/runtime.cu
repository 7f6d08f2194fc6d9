// runtime.cu -- error plumbing and per-device launch prerequisites shared by the libdfthermo.so sources.
#include "common.cuh"

static thread_local char g_err[512] = "";

df_status df_set_error(df_status code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

extern "C" const char* df_last_error(void) { return g_err; }
extern "C" int df_abi_version(void) { return 2; }

df_status df_ensure_dyn_smem(const void* kernel, int bytes, DfPerDevice* state) {
    int dev = 0;
    DF_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 128) return df_set_error(DF_ERR_UNSUPPORTED, "device ordinal %d not supported", dev);
    std::atomic<unsigned long long>& word = state->done[dev >> 6];
    const unsigned long long bit = 1ull << (dev & 63);
    if (word.load(std::memory_order_acquire) & bit) return DF_OK;
    // idempotent: two threads racing here both set the same value
    DF_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    word.fetch_or(bit, std::memory_order_release);
    return DF_OK;
}

int df_device_sm_count() {
    static std::atomic<int> cache[128];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 128) return 0;
    int v = cache[dev].load(std::memory_order_relaxed);
    if (v > 0) return v;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    cache[dev].store(v, std::memory_order_relaxed);
    return v;
}
