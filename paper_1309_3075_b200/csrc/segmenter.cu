// a1: on-device epoch-boundary segmenter (PAPER.md L78 change-point process; L117 per-branch epoch weights).
//
// Epoch e covers heights [tau[e-1], tau[e]).  For a branch (h_child, h_parent]:
//   e_lo = #{k : tau_k <= h_child}     epoch that holds the child end
//   e_hi = #{k : tau_k <  h_parent}    epoch that holds the parent end        (reading A3)
// Segments run e_hi, e_hi-1, ..., e_lo (parent end first, Eq. 5-7 / reading A2); every duration is > 0 because
// tau is strictly increasing and tau[e_hi-1] < h_parent, tau[e_lo] > h_child.  A zero-length branch has no segment.
//
// Three kernels: count (binary searches) -> single-CTA scan + counting sort by n_seg (longest first, the launch
// order of the chain kernels) -> fill (CSR epoch / duration arrays).
#include "epx_internal.h"
#include "seg_common.cuh"

namespace {

using epxseg::count_less;
using epxseg::branch_ends;

__global__ void seg_count_kernel(int n_br, int M, const double* __restrict__ tau, const int32_t* __restrict__ parent,
                                 const double* __restrict__ height, const double* __restrict__ child_h,
                                 const double* __restrict__ parent_h, int32_t* __restrict__ n_seg,
                                 int32_t* __restrict__ e_hi_out)
{
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_br) return;
    double hc, hp;
    branch_ends(b, parent, height, child_h, parent_h, hc, hp);
    int e_lo = count_less(tau, M - 1, hc, true);
    int e_hi = count_less(tau, M - 1, hp, false);
    e_hi_out[b] = e_hi;
    n_seg[b] = (hp > hc) ? (e_hi - e_lo + 1) : 0;
}

// One CTA: exclusive scan of n_seg into seg_off, and a counting sort of the slots by n_seg, longest first.
__global__ void __launch_bounds__(1024) seg_scan_sort_kernel(int n_br, const int32_t* __restrict__ n_seg,
                                                             int32_t* __restrict__ seg_off, int32_t* __restrict__ order)
{
    __shared__ int warp_tot[32];
    __shared__ int carry;
    __shared__ int hist[EPX_SORT_BINS];
    __shared__ int bin_base[EPX_SORT_BINS];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry = 0;
    if (tid < EPX_SORT_BINS) hist[tid] = 0;
    __syncthreads();
    for (int base = 0; base < n_br; base += blockDim.x) {
        int i = base + tid;
        int v = i < n_br ? n_seg[i] : 0;
        if (i < n_br) atomicAdd(&hist[min(v, EPX_SORT_BINS - 1)], 1);
        int x = v;
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_tot[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int w = warp_tot[lane];
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += y;
            }
            warp_tot[lane] = w;   // inclusive over warps
        }
        __syncthreads();
        int prefix = carry + (wid ? warp_tot[wid - 1] : 0) + x - v;   // exclusive
        if (i < n_br) seg_off[i] = prefix;
        __syncthreads();
        if (tid == blockDim.x - 1) carry = prefix + v;
        __syncthreads();
    }
    if (tid == 0) {
        seg_off[n_br] = carry;
        int acc = 0;
        for (int k = EPX_SORT_BINS - 1; k >= 0; k--) { bin_base[k] = acc; acc += hist[k]; }
    }
    __syncthreads();
    for (int i = tid; i < n_br; i += blockDim.x) {
        int k = min(n_seg[i], EPX_SORT_BINS - 1);
        int pos = atomicAdd(&bin_base[k], 1);
        order[pos] = i;
    }
}

__global__ void seg_fill_kernel(int n_br, int M, const double* __restrict__ tau, const int32_t* __restrict__ parent,
                                const double* __restrict__ height, const double* __restrict__ child_h,
                                const double* __restrict__ parent_h, const int32_t* __restrict__ n_seg,
                                const int32_t* __restrict__ e_hi_in, const int32_t* __restrict__ seg_off,
                                const double* __restrict__ brate, int32_t* __restrict__ seg_epoch,
                                double* __restrict__ seg_dur)
{
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_br) return;
    int n = n_seg[b];
    if (n == 0) return;
    double hc, hp;
    branch_ends(b, parent, height, child_h, parent_h, hc, hp);
    int e = e_hi_in[b], off = seg_off[b];
    const double rv = brate ? brate[b] : 1.0;      // branch rate scalar r_v, constant along the branch
    double upper = hp;
    for (int i = 0; i < n; i++, e--) {
        double lower = (i == n - 1) ? hc : tau[e - 1];
        seg_epoch[off + i] = e;
        seg_dur[off + i] = brate ? (upper - lower) * rv : upper - lower;
        upper = lower;
    }
}

// All three steps in ONE CTA for small problems (configs 1 and 3; many small instances batched): three dependent launches
// of a few microseconds each cost more in launch gaps than in work.  Pass 1 per chunk of 1024 slots: binary searches, block
// scan of the segment counts, each thread fills its own branch's segments.  Pass 2: counting sort by chain length.
constexpr int SEG_FUSED_MAX = 2048;     // beyond two chunks the single CTA loses to three parallel launches (cfg 2: 20 vs 18 us; cfg 5: 113 vs 33 us)

__global__ void __launch_bounds__(1024) seg_fused_kernel(int n_br, int M, const double* __restrict__ tau,
    const int32_t* __restrict__ parent, const double* __restrict__ height, const double* __restrict__ child_h,
    const double* __restrict__ parent_h, const double* __restrict__ brate, int32_t* __restrict__ n_seg,
    int32_t* __restrict__ e_hi_out, int32_t* __restrict__ seg_off, int32_t* __restrict__ seg_epoch,
    double* __restrict__ seg_dur, int32_t* __restrict__ order)
{
    __shared__ int warp_tot[32];
    __shared__ int carry;
    __shared__ int hist[EPX_SORT_BINS];
    __shared__ int bin_base[EPX_SORT_BINS];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry = 0;
    if (tid < EPX_SORT_BINS) hist[tid] = 0;
    __syncthreads();
    for (int base = 0; base < n_br; base += 1024) {
        const int b = base + tid;
        int v = 0, e_hi = 0;
        double hc = 0.0, hp = 0.0;
        if (b < n_br) {
            branch_ends(b, parent, height, child_h, parent_h, hc, hp);
            const int e_lo = count_less(tau, M - 1, hc, true);
            e_hi = count_less(tau, M - 1, hp, false);
            v = (hp > hc) ? (e_hi - e_lo + 1) : 0;
            e_hi_out[b] = e_hi;
            n_seg[b] = v;
            atomicAdd(&hist[min(v, EPX_SORT_BINS - 1)], 1);
        }
        int x = v;
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_tot[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int w = warp_tot[lane];
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += y;
            }
            warp_tot[lane] = w;   // inclusive over warps
        }
        __syncthreads();
        const int off = carry + (wid ? warp_tot[wid - 1] : 0) + x - v;   // exclusive prefix
        if (b < n_br) {
            seg_off[b] = off;
            const double rv = brate ? brate[b] : 1.0;
            double upper = hp;
            int e = e_hi;
            for (int i = 0; i < v; i++, e--) {
                const double lower = (i == v - 1) ? hc : tau[e - 1];
                seg_epoch[off + i] = e;
                seg_dur[off + i] = brate ? (upper - lower) * rv : upper - lower;
                upper = lower;
            }
        }
        __syncthreads();
        if (tid == 1023) carry = off + v;
        __syncthreads();
    }
    if (tid == 0) {
        seg_off[n_br] = carry;
        int acc = 0;
        for (int k = EPX_SORT_BINS - 1; k >= 0; k--) { bin_base[k] = acc; acc += hist[k]; }
    }
    __syncthreads();
    for (int i = tid; i < n_br; i += 1024) {
        const int k = min(n_seg[i], EPX_SORT_BINS - 1);
        order[atomicAdd(&bin_base[k], 1)] = i;
    }
}

}  // namespace

int launch_segmenter(const epx_ctx* c, cudaStream_t s)
{
    const DevBuffers& d = c->d;
    int n = c->n_slots;
    int blocks = (n + 255) / 256;
    const int32_t* parent = c->tree_mode ? d.parent : nullptr;
    if (n <= SEG_FUSED_MAX) {
        seg_fused_kernel<<<1, 1024, 0, s>>>(n, c->M, d.tau, parent, d.height, d.child_h, d.parent_h, c->has_brates ? d.brate : nullptr,
                                            d.n_seg, d.e_hi, d.seg_off, d.seg_epoch, d.seg_dur, d.order);
        return cudaGetLastError() == cudaSuccess ? 1 : -1;
    }
    seg_count_kernel<<<blocks, 256, 0, s>>>(n, c->M, d.tau, parent, d.height, d.child_h, d.parent_h, d.n_seg, d.e_hi);
    seg_scan_sort_kernel<<<1, 1024, 0, s>>>(n, d.n_seg, d.seg_off, d.order);
    seg_fill_kernel<<<blocks, 256, 0, s>>>(n, c->M, d.tau, parent, d.height, d.child_h, d.parent_h, d.n_seg, d.e_hi,
                                           d.seg_off, c->has_brates ? d.brate : nullptr, d.seg_epoch, d.seg_dur);
    return cudaGetLastError() == cudaSuccess ? 3 : -1;
}

// ---------------------------------------------------------------------------------------------------------------------------
// epx_segment_branches_static: a1 for callers that have no device memory to lend (include/epx.h has the contract).
//
// Every other path of the library carves its intermediates (n_seg, e_hi, order above) out of the workspace the caller binds.
// Here the same three intermediates sit in ONE array that is part of the library's device image, so the call needs the
// caller's inputs and outputs and nothing else: no cudaMalloc, no workspace, no context object.
//
// What is easy to get wrong, and is therefore kept in this one file:
//   - In HOST code `g_static_seg_scratch` is only the handle the runtime registered for the symbol.  It is not a device
//     address; a kernel handed `g_static_seg_scratch` from the host would fault (or, on a system where the GPU can reach host
//     memory, quietly scribble somewhere else).  The device address is asked for with cudaGetSymbolAddress, once per device,
//     while that device is current, and that pointer is what the kernels get.
//   - Each device that loads the library has its own copy of the array at its own address, hence the per-device table.
//   - The array outlives every call and keeps what the last call left in it.  Nothing below reads a word before the same call
//     has written it (count writes n_seg / e_hi for [0, n_br), scan + sort writes order for [0, n_br), fill reads only those),
//     so nothing has to be cleared -- a future user of this array that accumulates into it must clear its part first.
// ---------------------------------------------------------------------------------------------------------------------------
#include <mutex>
#include <stdio.h>
#include "../../include/epx.h"

// n_seg | e_hi | order, EPX_STATIC_MAX_BRANCHES entries each: 3 * 32768 * 4 B = 384 KiB per device, held until the process exits.
static __device__ __align__(256) int32_t g_static_seg_scratch[3 * EPX_STATIC_MAX_BRANCHES];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
int32_t* g_static_scratch_addr[STATIC_MAX_DEVICES];   // device address of the array on device i; nullptr = not looked up yet
std::mutex g_static_mu;

// The fill step of a1 with the caller's capacity respected: segments whose position is >= cap are not stored (the caller
// sees the shortfall in seg_off[n_br]).  Same expressions as seg_fill_kernel, so the stored values have the same bits.
__global__ void seg_fill_capped_kernel(int n_br, const double* __restrict__ tau, const double* __restrict__ child_h,
                                       const double* __restrict__ parent_h, const int32_t* __restrict__ n_seg,
                                       const int32_t* __restrict__ e_hi_in, const int32_t* __restrict__ seg_off, int cap,
                                       int32_t* __restrict__ seg_epoch, double* __restrict__ seg_dur)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_br) return;
    const int n = n_seg[b];
    if (n == 0) return;
    const double hc = child_h[b], hp = parent_h[b];
    int e = e_hi_in[b];
    const int off = seg_off[b];
    double upper = hp;
    for (int i = 0; i < n; i++, e--) {
        const double lower = (i == n - 1) ? hc : tau[e - 1];
        if (off + i < cap) {
            seg_epoch[off + i] = e;
            seg_dur[off + i] = upper - lower;
        }
        upper = lower;
    }
}

int static_fail(char* errbuf, size_t errbuf_len, int code, const char* what, const char* detail = nullptr)
{
    if (errbuf && errbuf_len) snprintf(errbuf, errbuf_len, detail ? "epx_segment_branches_static: %s (%s)" : "epx_segment_branches_static: %s", what, detail);
    return code;
}

}  // namespace

extern "C" int epx_segment_branches_static(int device, int n_br, int M, const double* dev_tau, const double* dev_child_height,
                                           const double* dev_parent_height, int32_t* dev_seg_off, int32_t* dev_seg_epoch,
                                           double* dev_seg_dur, int cap, void* cuda_stream, char* errbuf, size_t errbuf_len)
{
    if (errbuf && errbuf_len) errbuf[0] = 0;
    // argument checks first: none of them touches the CUDA runtime
    if (n_br > EPX_STATIC_MAX_BRANCHES) {
        char msg[160];
        snprintf(msg, sizeof msg, "n_br = %d exceeds EPX_STATIC_MAX_BRANCHES = %d, the size of the built-in scratch array; "
                 "split the branch list or use a bound context", n_br, EPX_STATIC_MAX_BRANCHES);
        return static_fail(errbuf, errbuf_len, EPX_E_WORKSPACE, msg);
    }
    if (n_br < 0 || M < 1 || M > EPX_MAX_M || cap < 0 || device < 0 || device >= STATIC_MAX_DEVICES)
        return static_fail(errbuf, errbuf_len, EPX_E_ARG, "n_br, M, cap or device out of range");
    if (!dev_seg_off || (M > 1 && !dev_tau) || (n_br > 0 && (!dev_child_height || !dev_parent_height)) ||
        (cap > 0 && (!dev_seg_epoch || !dev_seg_dur)))
        return static_fail(errbuf, errbuf_len, EPX_E_ARG, "a required device pointer is NULL");

    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
    if (e != cudaSuccess) return static_fail(errbuf, errbuf_len, EPX_E_CUDA, "cannot select the device", cudaGetErrorString(e));

    // set-up, once per device, with that device current: where does this device keep the array?
    int32_t* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_scratch_addr[device]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_seg_scratch);
            if (e == cudaSuccess && !p) e = cudaErrorInvalidSymbol;
            if (e == cudaSuccess) g_static_scratch_addr[device] = static_cast<int32_t*>(p);
        }
        scratch = g_static_scratch_addr[device];
    }
    int rc = EPX_OK;
    if (e != cudaSuccess) {
        rc = static_fail(errbuf, errbuf_len, EPX_E_CUDA, "cudaGetSymbolAddress of the scratch array failed", cudaGetErrorString(e));
    } else {
        int32_t* n_seg = scratch;
        int32_t* e_hi = scratch + EPX_STATIC_MAX_BRANCHES;
        int32_t* order = scratch + 2 * EPX_STATIC_MAX_BRANCHES;
        cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
        const int blocks = (n_br + 255) / 256;
        if (n_br > 0)
            seg_count_kernel<<<blocks, 256, 0, s>>>(n_br, M, dev_tau, nullptr, nullptr, dev_child_height, dev_parent_height, n_seg, e_hi);
        seg_scan_sort_kernel<<<1, 1024, 0, s>>>(n_br, n_seg, dev_seg_off, order);   // n_br == 0: writes seg_off[0] = 0 only
        if (n_br > 0)
            seg_fill_capped_kernel<<<blocks, 256, 0, s>>>(n_br, dev_tau, dev_child_height, dev_parent_height, n_seg, e_hi, dev_seg_off,
                                                          cap, dev_seg_epoch, dev_seg_dur);
        e = cudaGetLastError();
        if (e != cudaSuccess) rc = static_fail(errbuf, errbuf_len, EPX_E_CUDA, "kernel launch failed", cudaGetErrorString(e));
    }
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    return rc;
}
