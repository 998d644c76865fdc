// sc_static.cu -- sc_neighbour_counts_static: the neighbour count of a plan (the verification pass of
// sc_debug_neighbour_counts) for callers that must not allocate: code under CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc.  For a NESTED plan the count kernel writes RING-ordered counts and signatures to
// scratch memory and a second kernel gathers them into the caller's NESTED-ordered outputs; sc_debug_neighbour_counts
// takes that scratch from cudaMalloc / cudaFree on every call, this entry point takes it from a file-scope __device__
// array of fixed size (every GPU that loads libsc holds its SC_STATIC_MAX_NPIX x 12 bytes = 2.25 MiB until exit).
//
// The array's name is a device symbol: in HOST code it is a stand-in, not a device address.  Its address is resolved
// here, once per device with that device current, by cudaGetSymbolAddress, and the resolved pointer is what the
// kernels get.
//
// Every call shares the array and the array keeps the last call's contents.  Nothing has to start at zero: the count
// kernel overwrites entries [0, N_pix) of both parts before the gather reads them, in stream order.  Two calls that
// overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it: serialise them.
#include "../../include/sc.h"
#include "sc_internal.cuh"

#include <mutex>

struct sc_plan;

namespace sc {
cudaError_t launch_generic_count(const Dev &P, int *count_dev, unsigned long long *sig_dev, const Audit *au, cudaStream_t st);
cudaError_t reorder_i32(int nside, int dir, const int *src, int *dst, cudaStream_t st);
cudaError_t reorder_u64(int nside, int dir, const unsigned long long *src, unsigned long long *dst, cudaStream_t st);
const Dev *plan_dev(const sc_plan *plan);
int plan_nested(const sc_plan *plan);
int plan_device(const sc_plan *plan);
void note_error(const char *what, cudaError_t e);
void note_message(const char *msg);
}  // namespace sc

namespace {

constexpr size_t kMaxNpix = SC_STATIC_MAX_NPIX;
// [0, 8 kMaxNpix): RING-ordered signatures (u64); [8 kMaxNpix, 12 kMaxNpix): RING-ordered counts (i32)
static __device__ __align__(256) unsigned char g_scratch[kMaxNpix * 12];

constexpr int kMaxDevices = 64;
std::mutex g_mutex;
unsigned char *g_scratch_addr[kMaxDevices] = {};

// device address of g_scratch on `device`, which must be the current device (resolved on the first call per device)
sc_status scratch_address(int device, unsigned char **addr) {
    if (device < 0 || device >= kMaxDevices) return SC_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch_addr[device]) {
        int cur = -1;
        cudaError_t e = cudaGetDevice(&cur);
        if (e != cudaSuccess) { sc::note_error("cudaGetDevice", e); return SC_ERR_CUDA; }
        if (cur != device) {
            sc::note_message("sc_neighbour_counts_static: the plan's device must be the current device");
            return SC_ERR_INVALID_ARG;
        }
        unsigned char *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_scratch);
        if (e != cudaSuccess || !p) { sc::note_error("cudaGetSymbolAddress(g_scratch)", e); return SC_ERR_CUDA; }
        g_scratch_addr[device] = p;
    }
    *addr = g_scratch_addr[device];
    return SC_OK;
}

}  // namespace

extern "C" sc_status sc_neighbour_counts_static(const sc_plan *plan, int32_t *count_dev, uint64_t *sig_dev, void *cuda_stream) {
    if (!plan || !count_dev) return SC_ERR_INVALID_ARG;
    const sc::Dev &D = *sc::plan_dev(plan);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((size_t)D.npix > kMaxNpix) {
        sc::note_message("sc_neighbour_counts_static: 12 nside^2 exceeds SC_STATIC_MAX_NPIX entries of static scratch");
        return SC_ERR_UNSUPPORTED;
    }
    cudaError_t e;
    if (!sc::plan_nested(plan)) {                                    // RING plan: no scratch needed
        if ((e = sc::launch_generic_count(D, count_dev, (unsigned long long *)sig_dev, nullptr, st)) != cudaSuccess) {
            sc::note_error("count", e);
            return SC_ERR_CUDA;
        }
        return SC_OK;
    }
    unsigned char *scratch = nullptr;
    const sc_status rs = scratch_address(sc::plan_device(plan), &scratch);
    if (rs != SC_OK) return rs;
    unsigned long long *s_ring = reinterpret_cast<unsigned long long *>(scratch);
    int *c_ring = reinterpret_cast<int *>(scratch + 8 * kMaxNpix);
    if ((e = sc::launch_generic_count(D, c_ring, sig_dev ? s_ring : nullptr, nullptr, st)) != cudaSuccess ||
        (e = sc::reorder_i32(D.nside, 1, c_ring, count_dev, st)) != cudaSuccess ||
        (sig_dev && (e = sc::reorder_u64(D.nside, 1, s_ring, (unsigned long long *)sig_dev, st)) != cudaSuccess)) {
        sc::note_error("sc_neighbour_counts_static launch", e);
        return SC_ERR_CUDA;
    }
    return SC_OK;
}
