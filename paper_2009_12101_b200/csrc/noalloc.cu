// noalloc.cu -- cbgmres_k_multidot_noalloc: the multi-dot S2 (Fig. 1 l.5) for callers that cannot
// allocate device memory (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
//
// The ordinary hook, cbgmres_k_multidot, needs a handle, and cbgmres_create allocates the scratch the pass
// reduces through (CTA partial sums, the last-block-done ticket).  Here that scratch is a file-scope device
// array of fixed size: every GPU that loads the library holds kNoAllocBytes (~ 0.6 MB) until the process exits.
// The kernels are the ordinary ones (launch_multidot, orth.cu) -- only the scratch pointers differ -- so the
// result has the bits of cbgmres_k_multidot's.
//
// In HOST code the array's name is a host-side stand-in, not a device address; the address the kernels get
// comes from cudaGetSymbolAddress, taken once per device with that device current (noalloc_setup below).
//
// The entry point calls no cudaMalloc / cudaFree / allocating library routine: it encodes tensor maps on the
// host (into thread-local storage), clears the control block with cudaMemsetAsync and launches.  Every call
// shares the one array per device and the array keeps the last call's contents; what must start at zero (the
// control block with the ticket) is cleared on the caller's stream before the launch.  Calls that overlap on one
// GPU (two streams, two host threads) race on the partial sums: callers serialise them.
#include "internal.cuh"

#include <mutex>
#include <stdio.h>

namespace {

using namespace cbg;

constexpr size_t kCtlBytes = (sizeof(Ctl) + 255) & ~size_t(255);
constexpr size_t kPartialsBytes = (size_t)kNumSMs * kLdp * sizeof(double);  // every pass runs at most kNumSMs CTAs
constexpr size_t kNpartBytes = (size_t)2 * kMaxGrid * sizeof(double);       // indexed [blockIdx] and [kMaxGrid + blockIdx]
constexpr size_t kNoAllocBytes = kCtlBytes + kPartialsBytes + kNpartBytes;
static_assert(kNoAllocBytes == CBGMRES_NOALLOC_SCRATCH_BYTES, "include/cbgmres.h states the size of the static scratch");
static_assert(kCtlBytes % 256 == 0 && kPartialsBytes % 8 == 0, "alignment of the scratch regions");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char *g_dev_ptr[kMaxDevices] = {}; // device address of g_noalloc_scratch on device d (null = not set up)
thread_local char g_err[256] = "";

int fail(int code, const char *msg)
{
    snprintf(g_err, sizeof g_err, "%s", msg);
    return code;
}

int fail_cuda(const char *what, cudaError_t e)
{
    snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
    return CBGMRES_E_CUDA;
}

inline int fmt_bytes_or_neg(int f)
{
    switch (f) {
    case CBGMRES_FP64: return 8;
    case CBGMRES_FP32: case CBGMRES_INT32: return 4;
    case CBGMRES_FP16: case CBGMRES_INT16: return 2;
    default: return -1;
    }
}

// Once per device, with that device current: the device address of the static array.
int noalloc_setup(int device, unsigned char **out)
{
    if (device < 0 || device >= kMaxDevices) return fail(CBGMRES_E_INVALID, "device index out of range");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_dev_ptr[device]) {
        int prev = -1;
        cudaError_t e = cudaGetDevice(&prev);
        if (e != cudaSuccess) return fail_cuda("cudaGetDevice", e);
        if (prev != device && (e = cudaSetDevice(device)) != cudaSuccess) return fail_cuda("cudaSetDevice", e);
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (prev != device) cudaSetDevice(prev);
        if (e != cudaSuccess) return fail_cuda("cudaGetSymbolAddress(g_noalloc_scratch)", e);
        if (!p || reinterpret_cast<uintptr_t>(p) % 256 != 0) return fail(CBGMRES_E_CUDA, "static scratch: bad device address");
        g_dev_ptr[device] = static_cast<unsigned char *>(p);
    }
    if (out) *out = g_dev_ptr[device];
    return CBGMRES_OK;
}

} // namespace

extern "C" {

const char *cbgmres_noalloc_last_error(void) { return g_err; }

int cbgmres_noalloc_setup(int32_t device) { return noalloc_setup(device, nullptr); }

int cbgmres_k_multidot_noalloc(int32_t device, void *stream, int32_t format, int64_t n, int64_t ld, int32_t k,
                               const void *d_V, const double *d_scales, const double *d_w, double *d_h)
{
    const int B = fmt_bytes_or_neg(format);
    if (B < 0) return fail(CBGMRES_E_INVALID, "unknown storage format");
    if (n <= 0 || ld < n || k < 0) return fail(CBGMRES_E_INVALID, "bad n / ld / k");
    if (k > CBGMRES_NOALLOC_MAX_K) {
        snprintf(g_err, sizeof g_err, "k = %d exceeds the static scratch of the no-allocation entry point (at most %d vectors per call)",
                 (int)k, CBGMRES_NOALLOC_MAX_K);
        return CBGMRES_E_INVALID;
    }
    if (!d_V || !d_w || !d_h) return fail(CBGMRES_E_INVALID, "null pointer argument");
    if (((size_t)ld * (size_t)B) % 16 != 0 || reinterpret_cast<uintptr_t>(d_V) % 16 != 0)
        return fail(CBGMRES_E_INVALID, "basis vectors must be 16-byte aligned (ld*bytes % 16 == 0)");
    if ((format == CBGMRES_INT32 || format == CBGMRES_INT16) && !d_scales)
        return fail(CBGMRES_E_INVALID, "fixed-point formats need d_scales");
    if (k == 0) return CBGMRES_OK;

    unsigned char *base = nullptr;
    const int rc = noalloc_setup(device, &base);
    if (rc) return rc;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return fail_cuda("cudaSetDevice", e);
    cudaStream_t s = static_cast<cudaStream_t>(stream);

    // the array keeps the last call's contents: the control block (ticket of the last-block-done stage, hook outputs)
    // starts from zero; the partial sums are written by every CTA before the final stage reads them
    e = cudaMemsetAsync(base, 0, kCtlBytes, s);
    if (e != cudaSuccess) return fail_cuda("cudaMemsetAsync(control block)", e);

    LaunchCtx lc;
    lc.device = device;
    lc.use_pdl = 0; // the predecessor on the stream is the memset above: plain stream order
    Scratch sc;
    sc.ctl = reinterpret_cast<Ctl *>(base);
    sc.partials = reinterpret_cast<double *>(base + kCtlBytes);
    sc.npart = reinterpret_cast<double *>(base + kCtlBytes + kPartialsBytes);
    sc.lc = &lc;
    BasisView bv{d_V, ld, d_scales, format};
    const int launched = launch_multidot(s, sc, bv, n, k, d_w, d_h, nullptr, MODE_HOOK, 0, 0);
    if (lc.orth_error) {
        snprintf(g_err, sizeof g_err, "tensor-map encode failed (CUresult %d)", lc.orth_error);
        return CBGMRES_E_CUDA;
    }
    if (lc.launch_error != cudaSuccess) {
        snprintf(g_err, sizeof g_err, "launch of %s failed: %s", lc.launch_kernel, cudaGetErrorString(lc.launch_error));
        return CBGMRES_E_CUDA;
    }
    if (launched < 1) return fail(CBGMRES_E_CUDA, "nothing was launched");
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda("launch", e);
    return CBGMRES_OK;
}

} // extern "C"
