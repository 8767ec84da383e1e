// sable_injections_static: the Step-2 recovery kernel (PAPER.md:80 eq. 5, :95-99 eq. 9; k_recover in sable_kernels2.cuh)
// for callers that may not allocate: no context, no cudaMalloc / cudaFree, no allocating library routine.  The kernel's
// scratch -- the voltages in rectangular form, one [n_bus] slice per scenario, which k_recover keeps in shared memory or in
// the context's workspace -- lives in ONE file-scope __device__ array of kStaticScratchBytes that every GPU loading the
// library holds until exit.  Every call (from any thread, on any stream) shares that array: calls that overlap on the GPU
// race on it; the array keeps the last call's contents, and nothing in it has to start at zero (each CTA writes its slice
// before it reads it).  This file shares no code path with the rest of the library.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/sable.h"

namespace {

constexpr size_t kStaticScratchBytes = SABLE_STATIC_SCRATCH_BYTES;       // 8 MiB: batch * n_bus <= 524 288 voltages
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// In host code `g_static_scratch` is only a handle for the runtime, not a device address: the address is looked up once per
// device (with that device current) and cached here.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char* g_scratch_ptr[kMaxDevices] = {};

struct StaticArgs {
    int32_t n_bus, batch;
    const int32_t *row_ptr, *col_idx;      // Y_bus CSR as the caller gives it (any column order, duplicates allowed: they add up)
    const double *y_re, *y_im;
    const double *vm, *va;                 // [batch][n_bus]
    double *p_inj, *q_inj;                 // [batch][n_bus]
    double2* scratch;                      // [batch][n_bus] rectangular voltages (the static array)
};

// One CTA per scenario, as k_recover: V = Vm e^{j theta} of the scenario into its scratch slice, then one Y_bus row per
// thread: S_i = V_i conj(sum_k Y_ik V_k).
__global__ void k_recover_static(const StaticArgs A) {
    const int b = blockIdx.x;
    const size_t o = (size_t)b * A.n_bus;
    double2* v = A.scratch + o;
    for (int i = threadIdx.x; i < A.n_bus; i += blockDim.x) {
        double sn, cs;
        sincos(A.va[o + i], &sn, &cs);
        const double m = A.vm[o + i];
        v[i] = make_double2(m * cs, m * sn);
    }
    __syncthreads();                        // the slice is written and read by this CTA only
    for (int i = threadIdx.x; i < A.n_bus; i += blockDim.x) {
        double ire = 0.0, iim = 0.0;
        const int k1 = A.row_ptr[i + 1];
        for (int k = A.row_ptr[i]; k < k1; ++k) {
            const double g = A.y_re[k], bb = A.y_im[k];
            const double2 x = v[A.col_idx[k]];
            ire += g * x.x - bb * x.y;
            iim += bb * x.x + g * x.y;
        }
        const double2 vi = v[i];
        A.p_inj[o + i] = vi.x * ire + vi.y * iim;
        A.q_inj[o + i] = vi.y * ire - vi.x * iim;
    }
}

sable_status report(char* errbuf, int32_t errbuf_len, sable_status s, const char* msg) {
    if (errbuf && errbuf_len > 0) snprintf(errbuf, (size_t)errbuf_len, "%s", msg);
    return s;
}

}  // namespace

extern "C" sable_status sable_injections_static(int32_t n_bus, int32_t batch, const int32_t* row_ptr, const int32_t* col_idx,
                                                const double* y_re, const double* y_im, const double* vm, const double* va,
                                                double* p_inj, double* q_inj, void* cuda_stream, char* errbuf,
                                                int32_t errbuf_len) {
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (n_bus < 1 || batch < 0) return report(errbuf, errbuf_len, SABLE_ERR_INVALID_ARG, "n_bus must be >= 1 and batch >= 0");
    if ((unsigned long long)n_bus * (unsigned long long)batch * sizeof(double2) > kStaticScratchBytes) {
        char msg[256];
        snprintf(msg, sizeof msg, "batch * n_bus = %lld voltages exceed the static scratch array (%lld voltages, %lld bytes): split the "
                 "batch or use sable_recover", (long long)n_bus * batch, (long long)(kStaticScratchBytes / sizeof(double2)), (long long)kStaticScratchBytes);
        return report(errbuf, errbuf_len, SABLE_ERR_INVALID_ARG, msg);
    }
    // set-up, once per device: the device address of the scratch array
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return report(errbuf, errbuf_len, SABLE_ERR_CUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return report(errbuf, errbuf_len, SABLE_ERR_CUDA, "device index beyond the per-device table of 64");
    unsigned char* ptr = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_scratch_ptr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess || !p) return report(errbuf, errbuf_len, SABLE_ERR_CUDA, e != cudaSuccess ? cudaGetErrorString(e) : "cudaGetSymbolAddress returned null");
            g_scratch_ptr[dev] = static_cast<unsigned char*>(p);
        }
        ptr = g_scratch_ptr[dev];
    }
    if (batch == 0) return SABLE_OK;         // set-up only
    if (!row_ptr || !col_idx || !y_re || !y_im || !vm || !va || !p_inj || !q_inj)
        return report(errbuf, errbuf_len, SABLE_ERR_INVALID_ARG, "null array");
    StaticArgs A{};
    A.n_bus = n_bus; A.batch = batch; A.row_ptr = row_ptr; A.col_idx = col_idx; A.y_re = y_re; A.y_im = y_im;
    A.vm = vm; A.va = va; A.p_inj = p_inj; A.q_inj = q_inj; A.scratch = reinterpret_cast<double2*>(ptr);
    const int th = n_bus <= 256 ? 64 : n_bus <= 4096 ? 256 : 512;
    k_recover_static<<<batch, th, 0, (cudaStream_t)cuda_stream>>>(A);
    e = cudaGetLastError();
    if (e != cudaSuccess) return report(errbuf, errbuf_len, SABLE_ERR_CUDA, cudaGetErrorString(e));
    return SABLE_OK;
}
