// wpccc_cross_sections_static (include/wpccc.h): the cross-section integral of P:L106 (sigma = 2 pi Int b P(b) db, trapezoid
// rule in ln b) for callers that may not allocate device memory and hold no basis handle or
// workspace.  Same arithmetic as the sigma_* outputs of wpccc_probabilities (api.cu, k_cross_sections), but the index scratch
// (impact parameters, the order of the trajectories sorted by b inside each velocity group, the group offsets) lives in
// the file-scope device array below instead of the basis arena.
//
// The array is part of the library image: every GPU that loads libwpccc.so holds WPCCC_STATIC_SCRATCH_BYTES (256 KiB)
// from the first CUDA call until the process exits.  Every call on a device uses the same array, so two calls whose GPU
// work overlaps (different streams, different host threads) race; one call at a time per device.  The array keeps the last
// call's contents: a call writes every element its kernel reads (b[0..n), order[0..n), goff[0..n_vgroups]) before the
// launch, nothing relies on zero initial contents, and nothing past those ranges is read.
//
// In host code `g_static_scratch` is a host-side stand-in for the symbol, not a device address; the device address is
// asked for once per device, with that device current (cudaGetSymbolAddress), and handed to the kernel.
// No cudaMalloc / cudaFree / allocating library routine is called here.
#include <algorithm>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace {

static __device__ __align__(256) unsigned char g_static_scratch[WPCCC_STATIC_SCRATCH_BYTES];

std::mutex g_static_mu;
unsigned char *g_static_ptr[64] = {nullptr};          // per device ordinal: device address of g_static_scratch

// device address of the scratch array on the current device (looked up once per device)
int static_scratch(unsigned char **out) {
    int dev = 0;
    WP_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) WP_FAIL(WPCCC_EINVAL, "device ordinal %d outside 0..63", dev);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        unsigned char *p = nullptr;
        WP_CUDA(cudaGetSymbolAddress((void **)&p, g_static_scratch));
        if (!p || (reinterpret_cast<size_t>(p) & 255)) WP_FAIL(WPCCC_ECUDA, "static scratch: bad device address %p", (void *)p);
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return 0;
}

// the layout of one call inside the array
struct StaticLayout {
    size_t off_b, off_order, off_goff, bytes;
    StaticLayout(int n_traj, int n_vgroups) {
        off_b = 0;
        off_order = (off_b + (size_t)n_traj * sizeof(double) + 255) & ~(size_t)255;
        off_goff = (off_order + (size_t)n_traj * sizeof(int) + 255) & ~(size_t)255;
        bytes = off_goff + ((size_t)n_vgroups + 1) * sizeof(int);
    }
};

// sigma[g][col] = 2 pi sum over consecutive (sorted by b) pairs of 0.5 dln(b) (b0^2 P0 + b1^2 P1); scratch = the static array
__global__ void k_cross_sections_static(const double *P, int ncol, const unsigned char *scratch, size_t off_order, size_t off_goff, double *sigma) {
    const double *b = reinterpret_cast<const double *>(scratch);
    const int *order = reinterpret_cast<const int *>(scratch + off_order), *goff = reinterpret_cast<const int *>(scratch + off_goff);
    const int g = blockIdx.x;
    for (int col = blockIdx.y * blockDim.x + threadIdx.x; col < ncol; col += gridDim.y * blockDim.x) {
        double s = 0.0;
        for (int k = goff[g]; k + 1 < goff[g + 1]; ++k) {
            const int t0 = order[k], t1 = order[k + 1];
            const double dl = log(b[t1]) - log(b[t0]);
            s += 2.0 * 3.14159265358979323846 * 0.5 * dl * (b[t0] * b[t0] * P[(size_t)t0 * ncol + col] + b[t1] * b[t1] * P[(size_t)t1 * ncol + col]);
        }
        sigma[(size_t)g * ncol + col] = s;
    }
}

}  // namespace

extern "C" int wpccc_cross_sections_static(int n_traj, int n_cols, const double *dP, const double *b, const int *vgroup, int n_vgroups,
                                           double *dSigma, void *stream) {
    if (!dP || !dSigma || !b || !vgroup) WP_FAIL(WPCCC_EINVAL, "cross_sections_static: dP / dSigma / b / vgroup NULL");
    if (n_traj < 1 || n_cols < 1 || n_vgroups < 1) WP_FAIL(WPCCC_EINVAL, "cross_sections_static: n_traj, n_cols, n_vgroups must be >= 1");
    if (n_traj > WPCCC_STATIC_MAX_TRAJ)
        WP_FAIL(WPCCC_ENOMEM, "cross_sections_static: %d trajectories exceed the static scratch (at most %d per call; use wpccc_probabilities or call per velocity group)",
                n_traj, WPCCC_STATIC_MAX_TRAJ);
    if (n_vgroups > WPCCC_STATIC_MAX_VGROUPS)
        WP_FAIL(WPCCC_ENOMEM, "cross_sections_static: %d velocity groups exceed the static scratch (at most %d per call)", n_vgroups, WPCCC_STATIC_MAX_VGROUPS);
    const StaticLayout L(n_traj, n_vgroups);
    if (L.bytes > (size_t)WPCCC_STATIC_SCRATCH_BYTES) WP_FAIL(WPCCC_ENOMEM, "cross_sections_static: %zu bytes of scratch needed, %d held", L.bytes, WPCCC_STATIC_SCRATCH_BYTES);
    for (int t = 0; t < n_traj; ++t) {
        if (!(b[t] > 0.0)) WP_FAIL(WPCCC_EINVAL, "cross_sections_static: b[%d] must be > 0 (trapezoid rule in ln b)", t);
        if (vgroup[t] < 0 || vgroup[t] >= n_vgroups) WP_FAIL(WPCCC_EINVAL, "cross_sections_static: vgroup[%d] out of range", t);
    }
    unsigned char *scratch = nullptr;
    if (int rc = static_scratch(&scratch)) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    // host index vectors: trajectories of each velocity group in ascending b (ties keep the caller's order)
    std::vector<int> order, goff, m;
    order.reserve(n_traj); goff.reserve((size_t)n_vgroups + 1);
    for (int g = 0; g < n_vgroups; ++g) {
        goff.push_back((int)order.size());
        m.clear();
        for (int t = 0; t < n_traj; ++t) if (vgroup[t] == g) m.push_back(t);
        std::stable_sort(m.begin(), m.end(), [&](int x, int y) { return b[x] < b[y]; });
        order.insert(order.end(), m.begin(), m.end());
    }
    goff.push_back((int)order.size());
    // every element the kernel reads is rewritten here; the rest of the array keeps whatever the last call left
    WP_CUDA(cudaMemcpyAsync(scratch + L.off_b, b, (size_t)n_traj * sizeof(double), cudaMemcpyHostToDevice, s));
    WP_CUDA(cudaMemcpyAsync(scratch + L.off_order, order.data(), (size_t)n_traj * sizeof(int), cudaMemcpyHostToDevice, s));
    WP_CUDA(cudaMemcpyAsync(scratch + L.off_goff, goff.data(), goff.size() * sizeof(int), cudaMemcpyHostToDevice, s));
    const int threads = 128;
    dim3 grid(n_vgroups, std::min((n_cols + threads - 1) / threads, 64));
    k_cross_sections_static<<<grid, threads, 0, s>>>(dP, n_cols, scratch, L.off_order, L.off_goff, dSigma);
    WP_CUDA(cudaGetLastError());
    WP_CUDA(cudaStreamSynchronize(s));     // the host index vectors must outlive the copies; the array is free for the next call
    return 0;
}
