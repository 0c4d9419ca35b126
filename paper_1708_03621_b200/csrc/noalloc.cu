// jdft_overlap_noalloc: the subspace overlap M = C1^+ O C2 for callers that may not allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc) and therefore cannot hand the library a workspace.
//
// The overlap is the split-K complex FP64 GEMM of gemm.cu (k_gemm_dotk + the fixed-order k_splitk_reduce); its split-K
// partials are the one piece of scratch memory it needs.  Here they live in a FILE-SCOPE device array of a fixed, modest
// size, so the call needs neither a workspace nor any allocation: every GPU that loads the library holds the
// JDFT_NOALLOC_SCRATCH_BYTES (16 MiB) of this array until the process exits.
//
// In host code the array's NAME is only a host-side stand-in, not a device address (a kernel given it would fault or, where
// the GPU can reach host memory, silently use the wrong memory).  The device address is taken once per device, with
// that device current, by cudaGetSymbolAddress (below) and passed to the kernels.
//
// Sharing: every call on a device uses the same array, which keeps the previous call's contents.  Nothing of it has to
// start at zero -- each split-K slice writes every entry of its partial result (tiles whose k range is empty write
// zeros) and the reduction reads only entries this call wrote -- so it is never cleared.  Two calls of one process
// that overlap on the same GPU (issued on different streams) RACE on the array: issue jdft_overlap_noalloc calls on ONE
// stream at a time per device.  (The array is per process and per device; other processes have their own.)
// The first call per device resolves the array's address (which may load the module): make it outside graph capture.
#include <mutex>
#include "jdft_internal.h"

#define JDFT_NOALLOC_SCRATCH_BYTES ((size_t)16 << 20)
#define JDFT_NOALLOC_MAX_ENTRIES 65536   /* nb1 * nb2 <= 65 536 (e.g. 256 x 256): at least 16 split-K slices fit */
#define JDFT_NOALLOC_MAX_DEVICES 64

static __device__ __align__(256) double g_noalloc_scratch[JDFT_NOALLOC_SCRATCH_BYTES / sizeof(double)];

namespace {

// device address of g_noalloc_scratch on `device`, resolved once per device with that device current
int noalloc_scratch(int device, void **out) {
    static std::mutex mu;
    static void *addr[JDFT_NOALLOC_MAX_DEVICES] = {nullptr};
    if (device < 0 || device >= JDFT_NOALLOC_MAX_DEVICES) return jdft_fail(JDFT_EINVAL, "overlap_noalloc: device index %d out of range", device);
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        int prev = -1;
        JDFT_CUDA(cudaGetDevice(&prev));
        if (prev != device) JDFT_CUDA(cudaSetDevice(device));
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (prev != device) cudaSetDevice(prev);
        if (e != cudaSuccess) return jdft_cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
        if (!p || (((uintptr_t)p) & 255)) return jdft_fail(JDFT_ECUDA, "overlap_noalloc: bad scratch address");
        addr[device] = p;
    }
    *out = addr[device];
    return JDFT_OK;
}

}  // namespace

extern "C" int jdft_overlap_noalloc(const jdft_basis *b, const double *C1, int nb1, const double *C2, int nb2, double *M,
                                    jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "overlap_noalloc: null basis");
    if (nb1 < 0 || nb2 < 0) return jdft_fail(JDFT_EINVAL, "overlap_noalloc: negative size");
    if ((int64_t)nb1 * nb2 > JDFT_NOALLOC_MAX_ENTRIES)
        return jdft_fail(JDFT_EINVAL, "overlap_noalloc: nb1 * nb2 = %lld exceeds the built-in scratch limit of %d entries "
                         "(16 MiB static array); use jdft_overlap with a caller workspace", (long long)nb1 * nb2, JDFT_NOALLOC_MAX_ENTRIES);
    if (nb1 == 0 || nb2 == 0) return JDFT_OK;
    if (!C1 || !C2 || !M) return jdft_fail(JDFT_EINVAL, "overlap_noalloc: null data pointer");
    if ((((uintptr_t)C1) | ((uintptr_t)C2) | ((uintptr_t)M)) & 15) return jdft_fail(JDFT_EINVAL, "overlap_noalloc: data pointer not 16-byte aligned");
    void *scratch = nullptr;
    int rc = noalloc_scratch(b->device, &scratch);
    if (rc) return rc;
    // M stored column-major nb1 x nb2 == row-major [nb2][nb1]:  M[bb][a] = Omega sum_n C2[bb][n] conj(C1[a][n])
    return jdft_gemm_dotk(b, C2, nb2, C1, nb1, b->nG, 1, b->volume, nullptr, M, scratch, JDFT_NOALLOC_SCRATCH_BYTES, (cudaStream_t)s);
}
