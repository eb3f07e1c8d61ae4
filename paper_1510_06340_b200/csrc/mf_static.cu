// mf_static.cu — mf_totals_static(): the conserved totals (Eq.1's conserved quantities summed over the grid) of a state given by DEVICE
// pointers, WITHOUT any allocation: for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses
// that forbid it).  mf_conserved_totals() keeps its per-block partial sums in a cudaMalloc'ed buffer of the context; this variant keeps them
// in the file-scope array below, which every GPU that loads the library holds until exit.
//
//   * Limit: MF_STATIC_MAX_CELLS = 2^24 cells (256^3, the metric's grid): 1024 blocks x 16384 cells per block; 5 x 1024 partial sums = 40 KB.
//   * The array's name is a host-side stand-in in host code, not a device address: its address is taken with cudaGetSymbolAddress once per
//     device, with that device current, and handed to the kernels.
//   * Every call shares the array and it keeps the last call's contents.  Nothing in it has to start at zero: a call writes every slot it
//     later reads (slot b of component q is written by block b before the finishing kernel, ordered behind it on the same stream, reads
//     slots 0..nblocks-1), so stale contents beyond nblocks are never looked at.  Calls that OVERLAP on the GPU (different streams, or
//     several host threads on the same device) race on the array: serialise them.
//   * No cudaMalloc, cudaFree or allocating library routine; two small kernel launches on the caller's stream; asynchronous.
#include "../../include/mustaforce.h"
#include <cuda_runtime.h>
#include <mutex>
#include <string>

namespace {

constexpr int SB_THREADS = 256;
constexpr int SB_MAX_BLOCKS = 1024;
constexpr long long SB_CELLS_PER_BLOCK = 16384;
constexpr long long SB_MAX_CELLS = SB_MAX_BLOCKS * SB_CELLS_PER_BLOCK;      // 2^24
static_assert(SB_MAX_CELLS == MF_STATIC_MAX_CELLS, "header and kernel disagree on the limit");

static __device__ __align__(256) double g_static_partials[5 * SB_MAX_BLOCKS];

struct Ptr5 { const double* q[5]; };

// block b: the sums of its 16384 consecutive cells, component by component, into scratch[q * SB_MAX_BLOCKS + b]
__global__ void __launch_bounds__(SB_THREADS) k_static_partials(Ptr5 U, long long n, double* __restrict__ scratch)
{
    const long long lo = (long long)blockIdx.x * SB_CELLS_PER_BLOCK;
    const long long hi = lo + SB_CELLS_PER_BLOCK < n ? lo + SB_CELLS_PER_BLOCK : n;
    double acc[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
    for (long long o = lo + threadIdx.x; o < hi; o += SB_THREADS)
#pragma unroll
        for (int v = 0; v < 5; ++v) acc[v] += U.q[v][o];
    __shared__ double s[5][SB_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) acc[v] += __shfl_xor_sync(0xffffffffu, acc[v], off);
        if (lane == 0) s[v][warp] = acc[v];
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0.0;
        for (int w = 0; w < SB_THREADS / 32; ++w) t += s[threadIdx.x][w];
        scratch[threadIdx.x * SB_MAX_BLOCKS + blockIdx.x] = t;
    }
}

// one block of 5 warps: warp q adds the nb partial sums of component q in a fixed order and writes scale * sum to out[q]
__global__ void __launch_bounds__(160) k_static_finish(const double* __restrict__ scratch, int nb, double scale, double* __restrict__ out)
{
    const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double t = 0.0;
    for (int b = lane; b < nb; b += 32) t += scratch[q * SB_MAX_BLOCKS + b];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
    if (lane == 0) out[q] = scale * t;
}

// the array's device address, looked up once per device (with that device current)
std::mutex g_addr_mutex;
double* g_addr[64];
bool g_addr_known[64];
thread_local std::string g_static_err;

int static_fail(int code, const std::string& msg) { g_static_err = msg; return code; }

} // namespace

extern "C" {

const char* mf_static_last_error(void) { return g_static_err.c_str(); }

int mf_totals_static(const double* E, const double* Mx, const double* My, const double* Mz, const double* R, long long ncells, double scale,
                     double* out5, void* cuda_stream)
{
    if (!E || !Mx || !My || !Mz || !R || !out5) return static_fail(MF_EINVAL, "mf_totals_static: null pointer");
    if (ncells < 1) return static_fail(MF_EINVAL, "mf_totals_static: ncells must be >= 1");
    if (ncells > SB_MAX_CELLS)
        return static_fail(MF_EINVAL, "mf_totals_static: " + std::to_string(ncells) + " cells exceed the static scratch's limit of " +
                                      std::to_string(SB_MAX_CELLS) + " (MF_STATIC_MAX_CELLS); use mf_conserved_totals");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return static_fail(MF_ECUDA, std::string("mf_totals_static: no CUDA device: ") + cudaGetErrorString(e)); }
    if (dev < 0 || dev >= 64) return static_fail(MF_EINVAL, "mf_totals_static: device ordinal beyond 63");
    double* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_addr_mutex);
        if (!g_addr_known[dev]) {
            double* p = nullptr;
            e = cudaGetSymbolAddress((void**)&p, g_static_partials);
            if (e != cudaSuccess || !p) {
                cudaGetLastError();
                return static_fail(MF_ECUDA, std::string("mf_totals_static: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e));
            }
            g_addr[dev] = p; g_addr_known[dev] = true;
        }
        scratch = g_addr[dev];
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nb = (int)((ncells + SB_CELLS_PER_BLOCK - 1) / SB_CELLS_PER_BLOCK);
    Ptr5 U; U.q[0] = E; U.q[1] = Mx; U.q[2] = My; U.q[3] = Mz; U.q[4] = R;
    k_static_partials<<<nb, SB_THREADS, 0, st>>>(U, ncells, scratch);
    k_static_finish<<<1, 160, 0, st>>>(scratch, nb, scale, out5);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(MF_ECUDA, std::string("mf_totals_static: kernel launch: ") + cudaGetErrorString(e));
    return MF_OK;
}

} // extern "C"
