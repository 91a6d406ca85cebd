// qmc_static.cu -- the batched hot path for callers that must not allocate device memory: the workspace of the fused kernels
// (tile-queue heads, plan tables, per-tile partial sums, per-shift means) lives in a file-scope device array of a fixed size
// instead of a buffer the caller allocated.  Same kernels, same arithmetic, same results as qmc_lattice_integrate_batch.
//
// The array's name is a host-side stand-in in host code: its device address is looked up with cudaGetSymbolAddress, once per
// device and with that device current, and only that address is ever handed to a kernel.
#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

#include "qmc_kernels.h"

namespace {

constexpr size_t kStaticScratchBytes = (size_t)QMC_STATIC_SCRATCH_BYTES;

// Every GPU that loads the library holds these 4 MiB until the process exits.  The contents survive from call to call; nothing
// in it needs clearing by hand: a call resets the tile-queue heads itself (stream-ordered, part of every batch call) and every
// partial-sum slot and every per-shift mean it reads is written by the same call first.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_addr[kMaxDevices];            // device address of g_static_scratch per device ordinal, nullptr = not looked up yet

// the scratch array's address on the current device; nullptr after a failure (text left for qmc_last_cuda_error)
void* scratch_on_current_device() {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        qmc::report_cuda_error(e != cudaSuccess ? e : cudaErrorInvalidDevice, "qmc_lattice_integrate_batch_static: no usable current device");
        return nullptr;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);           // the symbol, never its host-side address
        if (e != cudaSuccess || !p) {
            qmc::report_cuda_error(e != cudaSuccess ? e : cudaErrorInvalidSymbol, "cudaGetSymbolAddress(static scratch)");
            return nullptr;
        }
        g_scratch_addr[dev] = p;
    }
    return g_scratch_addr[dev];
}

}  // namespace

extern "C" {

size_t qmc_static_scratch_bytes(void) { return kStaticScratchBytes; }

int qmc_lattice_integrate_batch_static(int count, const qmc_problem* problems, double* out_means, double* out_errs,
                                       double* out_shift_means, void* cuda_stream) {
    if (count < 1) return QMC_ERR_N;
    if (!problems || !out_means || !out_errs) return QMC_ERR_NULL;
    const size_t need = qmc_workspace_bytes(count, problems);      // pure host function of the structs
    if (need == 0) {                                               // an invalid struct: report what is wrong with it
        const int st = qmc_plan_info(count, problems, nullptr, nullptr, nullptr);
        return st != QMC_OK ? st : QMC_ERR_WORKSPACE;
    }
    if (need > kStaticScratchBytes) {
        char msg[200];
        snprintf(msg, sizeof(msg),
                 "qmc_lattice_integrate_batch_static: the batch needs %zu bytes of workspace, the static scratch array holds %zu "
                 "(use qmc_lattice_integrate_batch with a workspace of your own)", need, kStaticScratchBytes);
        qmc::report_cuda_error(cudaErrorInvalidValue, msg);
        return QMC_ERR_WORKSPACE;
    }
    void* scratch = scratch_on_current_device();
    if (!scratch) return QMC_ERR_CUDA;
    return qmc_lattice_integrate_batch(count, problems, out_means, out_errs, out_shift_means, scratch, kStaticScratchBytes, cuda_stream);
}

}  // extern "C"
