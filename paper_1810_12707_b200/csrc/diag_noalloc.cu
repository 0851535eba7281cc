// diag_noalloc.cu — mhd_energy_means_noalloc(): the scalar diagnostics of a real-space state for callers that have no
// device memory to give the library (include/mhd.h, "Diagnostics without a workspace").
//
// Every other entry point of libmhd works inside a workspace that the caller allocates and hands to mhd_bind().  That
// suits a solver, but not a piece of code that is merely *handed* eight field pointers and asked "is this state still
// sane?": an in-situ monitor or a check-pointing hook called from somebody else's time loop, a plug-in running inside an
// application that took all of HBM for its own arena at start-up and offers no allocator to its plug-ins, or a health
// check that runs while another thread of the process is capturing a CUDA graph (cudaMalloc / cudaFree synchronise the
// device and are not allowed to interleave with a global-mode capture).  Such callers cannot call cudaMalloc and have no
// mhd_ctx, so they cannot produce the 80 KB of block partials that the two-stage reduction needs between its kernels.
//
// Here that scratch is a file-scope __device__ array: part of the library image, present on every GPU that loads
// libmhd.so from the moment the module is loaded until the process exits (80 KB per GPU).  The kernels are the
// ones mhd_diagnostics() runs (diag_stage1 / diag_stage2 of kernels_point.cu, through their launchers): same grid, same
// tree order, so the ten numbers are bit for bit those of mhd_diagnostics() on the same real-space arrays.
//
// The array's name is only a device address inside device code.  In host code `g_partials` is a host-side shadow
// symbol: handing `g_partials` itself to a kernel would make the kernel write through a host address (a fault, or on
// systems where the GPU can reach host memory a silent write to the wrong place).  The host therefore asks the runtime
// for the device address with cudaGetSymbolAddress(), once per device and with that device current, and passes that.
#include <mutex>
#include <cstdio>
#include <cstring>

#include "../../include/mhd.h"
#include "kernels.h"

namespace {

// 1024 blocks x 10 partial results (ke, me, ie, mass, mom x3, etot sums; rho, P minima) = 80 KB per GPU.
constexpr int NOALLOC_PARTIALS = 1024 * 10;
static __device__ __align__(256) double g_partials[NOALLOC_PARTIALS];

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_lock;
double* g_partials_addr[MAX_DEVICES] = {};   // device address of g_partials on device d (nullptr = not looked up yet)

int fail(int code, char* errbuf, size_t len, const char* what, const char* detail = nullptr) {
    if (errbuf && len) {
        if (detail) snprintf(errbuf, len, "mhd_energy_means_noalloc: %s: %s", what, detail);
        else snprintf(errbuf, len, "mhd_energy_means_noalloc: %s", what);
    }
    return code;
}

}  // namespace

extern "C" int mhd_energy_means_noalloc(long long n, double gamma, const double* const dev_U[8], double* dev_out,
                                        void* cuda_stream, char* errbuf, size_t errbuf_len) {
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (n <= 0) return fail(MHD_ERR_INVALID_ARG, errbuf, errbuf_len, "n must be positive");
    if (n > MHD_NOALLOC_MAX_POINTS)
        return fail(MHD_ERR_INVALID_ARG, errbuf, errbuf_len,
                    "n exceeds MHD_NOALLOC_MAX_POINTS (2^30 grid points = 1024^3, the largest grid of the library)");
    if (!(gamma > 1.0)) return fail(MHD_ERR_INVALID_ARG, errbuf, errbuf_len, "gamma must exceed 1");
    if (!dev_U || !dev_out) return fail(MHD_ERR_INVALID_ARG, errbuf, errbuf_len, "null argument");
    for (int f = 0; f < 8; ++f)
        if (!dev_U[f]) return fail(MHD_ERR_INVALID_ARG, errbuf, errbuf_len, "null field pointer");
    if (mhd::diag_partial_doubles() > NOALLOC_PARTIALS)   // the reduction's grid outgrew the static array: refuse, never overrun
        return fail(MHD_ERR_NOMEM, errbuf, errbuf_len, "static scratch smaller than the reduction's block partials");

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(MHD_ERR_CUDA, errbuf, errbuf_len, "cudaGetDevice", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(MHD_ERR_INVALID_ARG, errbuf, errbuf_len, "device ordinal above 63");

    // Set-up, first call on each device: look up where g_partials lives on the CURRENT device.
    double* part = nullptr;
    {
        std::lock_guard<std::mutex> guard(g_setup_lock);
        part = g_partials_addr[dev];
        if (!part) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_partials);
            if (e != cudaSuccess || !p)
                return fail(MHD_ERR_CUDA, errbuf, errbuf_len, "cudaGetSymbolAddress(g_partials)",
                            e != cudaSuccess ? cudaGetErrorString(e) : "null address");
            g_partials_addr[dev] = part = static_cast<double*>(p);
        }
    }

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // Stage 1 overwrites all 1024 x 10 partials (blocks without points store the neutral elements), so whatever the
    // previous call left in g_partials is never read: nothing has to be cleared first.
    mhd::launch_diag_partial(n, dev_U, gamma, part, /*accumulate=*/0, st);
    mhd::launch_diag_final(part, dev_out, 1.0 / (double)n, st);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MHD_ERR_CUDA, errbuf, errbuf_len, "kernel launch", cudaGetErrorString(e));
    return MHD_OK;
}
