// C-ABI entry points wpccc_matrix_elements, wpccc_propagate, wpccc_probabilities, wpccc_workspace_bytes,
// wpccc_fp64_peak: argument checking, workspace carving and launch orchestration only (include/wpccc.h).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <map>

#include "common.cuh"
#include "sweep.cuh"

namespace {

struct Carver {
    char *base; size_t cap, off = 0; bool ok = true;
    Carver(void *b, size_t c) : base((char *)b), cap(c) {}
    template <class T> T *take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T *p = reinterpret_cast<T *>(base + off);
        off += n * sizeof(T);
        if (off > cap) ok = false;
        return p;
    }
};

// a1 geometry: position p = g * n_idx + li  ->  z = z_min + 0.5 (i0 + li) h, R = hypot(b_g, z), ...
struct GeomOut { double *R, *cosT, *sinT, *theta, *z, *v; };
__global__ void k_geometry_grid(int n_g, int n_idx, const double *b, const double *v, long long i0, double z_min, double h, GeomOut o) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_g * n_idx) return;
    const int g = p / n_idx, li = p % n_idx;
    const double z = __dadd_rn(z_min, __dmul_rn(0.5 * (double)(i0 + li), h)), bb = b[g];
    const double R = hypot(bb, z);
    o.R[p] = R; o.cosT[p] = z / R; o.sinT[p] = bb / R; o.theta[p] = atan2(bb, z); o.z[p] = z; o.v[p] = v ? v[g] : 1.0;
}
__global__ void k_geometry_list(int n, const double *b, const double *z, const double *v, GeomOut o) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const double R = hypot(b[p], z[p]);
    o.R[p] = R; o.cosT[p] = z[p] / R; o.sinT[p] = b[p] / R; o.theta[p] = atan2(b[p], z[p]); o.z[p] = z[p]; o.v[p] = v[p];
}

// S and H outputs of wpccc_matrix_elements from the phase-free blocks.
struct ComposeArgs {
    const double *K; double *S; double *H; const double *z, *v;
    const int *st_rad_T, *st_rad_P; const double *eps_T, *eps_P;
    int NT, NP, phases;
};
__global__ void k_compose(const ComposeArgs a) {
    const int p = blockIdx.x, N = a.NT + a.NP;
    const double t = a.z[p] / a.v[p];
    for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < N * N; e += gridDim.y * blockDim.x) {
        const int i = e / N, j = e % N;
        double pr = 1.0, pi = 0.0;
        if (a.phases) {
            const double ei = (i < a.NT) ? a.eps_T[a.st_rad_T[i]] : a.eps_P[a.st_rad_P[i - a.NT]];
            const double ej = (j < a.NT) ? a.eps_T[a.st_rad_T[j]] : a.eps_P[a.st_rad_P[j - a.NT]];
            sincos((ei - ej) * t, &pi, &pr);
        }
        const size_t o = ((size_t)p * N * N + e) * 2;
        if (a.H) { const double hr = a.H[o], hi = a.H[o + 1]; a.H[o] = hr * pr - hi * pi; a.H[o + 1] = hr * pi + hi * pr; }
        if (a.S) {
            double sr = (i == j) ? 1.0 : 0.0, si = 0.0;
            if (a.NP > 0) {
                if (i >= a.NT && j < a.NT) { const double *k = a.K + (((size_t)p * a.NP + (i - a.NT)) * a.NT + j) * 2; sr = k[0]; si = k[1]; }
                else if (i < a.NT && j >= a.NT) { const double *k = a.K + (((size_t)p * a.NP + (j - a.NT)) * a.NT + i) * 2; sr = k[0]; si = -k[1]; }
            }
            a.S[o] = sr * pr - si * pi; a.S[o + 1] = sr * pi + si * pr;
        }
    }
}

__global__ void k_init_amplitudes(double *C, int n_traj, int N, int init_state) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (size_t)n_traj * N) return;
    C[2 * e] = ((int)(e % N) == init_state) ? 1.0 : 0.0; C[2 * e + 1] = 0.0;
}

// a9 observables
struct ProbArgs {
    const double *C; int n_traj, N, n_rad_tot;
    const int *st_rad_glob;          // [N] global radial index of each state
    const int *rad_class;            // [n_rad_tot] class 0..4
    double *P_state, *P_nl, *P_class;
};
__global__ void k_probabilities(const ProbArgs a) {
    const int t = blockIdx.x;
    extern __shared__ double sh[];   // [n_rad_tot]
    for (int r = threadIdx.x; r < a.n_rad_tot; r += blockDim.x) sh[r] = 0.0;
    __syncthreads();
    // one thread per radial function sums its m-substates in ascending order (deterministic)
    for (int j = threadIdx.x; j < a.N; j += blockDim.x) {
        const double *c = a.C + ((size_t)t * a.N + j) * 2;
        const double pj = c[0] * c[0] + c[1] * c[1];
        if (a.P_state) a.P_state[(size_t)t * a.N + j] = pj;
    }
    __syncthreads();
    for (int r = threadIdx.x; r < a.n_rad_tot; r += blockDim.x) {
        double s = 0.0;
        for (int j = 0; j < a.N; ++j) if (a.st_rad_glob[j] == r) { const double *c = a.C + ((size_t)t * a.N + j) * 2; s += c[0] * c[0] + c[1] * c[1]; }
        sh[r] = s;
        if (a.P_nl) a.P_nl[(size_t)t * a.n_rad_tot + r] = s;
    }
    __syncthreads();
    if (a.P_class && threadIdx.x < 5) {
        double s = 0.0;
        for (int r = 0; r < a.n_rad_tot; ++r) if (a.rad_class[r] == (int)threadIdx.x) s += sh[r];
        a.P_class[(size_t)t * 5 + threadIdx.x] = s;
    }
}
// sigma[g][col] = 2 pi sum over consecutive (sorted by b) pairs of 0.5 dln(b) (b0^2 P0 + b1^2 P1)
__global__ void k_cross_sections(const double *P, int ncol, const double *b, const int *order, const int *goff, double *sigma) {
    const int g = blockIdx.x;
    for (int col = threadIdx.x; col < ncol; col += blockDim.x) {
        double s = 0.0;
        for (int k = goff[g]; k + 1 < goff[g + 1]; ++k) {
            const int t0 = order[k], t1 = order[k + 1];
            const double dl = log(b[t1]) - log(b[t0]);
            s += 2.0 * 3.14159265358979323846 * 0.5 * dl * (b[t0] * b[t0] * P[(size_t)t0 * ncol + col] + b[t1] * b[t1] * P[(size_t)t1 * ncol + col]);
        }
        sigma[(size_t)g * ncol + col] = s;
    }
}

GeomOut carve_geom(Carver &cv, size_t n) {
    GeomOut g;
    g.R = cv.take<double>(n); g.cosT = cv.take<double>(n); g.sinT = cv.take<double>(n);
    g.theta = cv.take<double>(n); g.z = cv.take<double>(n); g.v = cv.take<double>(n);
    return g;
}

// elements of one block of positions (geometry already on the device): F, then H0 / K (two-centre) or Dre (one-centre)
int elements_two_centre(wpccc_basis *B, int n_pos, const GeomOut &g, double *d_F, double *d_K, double *d_H, void *tws, size_t tws_bytes,
                        int chunk, cudaStream_t s, const TransferSel *sel = nullptr) {
    const int NT = B->c[0].n_states, NP = B->c[1].n_states, N = NT + NP;
    int rc = wp_direct_gemm(B, n_pos, g.R, d_F, B->E_tot, s); if (rc) return rc;
    rc = wp_direct_assemble(B, 0, n_pos, g.cosT, d_F, B->E_tot, d_H, N, (long long)N * N, 1, s); if (rc) return rc;
    rc = wp_direct_assemble(B, 1, n_pos, g.cosT, d_F, B->E_tot, d_H + ((size_t)NT * N + NT) * 2, N, (long long)N * N, 1, s); if (rc) return rc;
    return wp_transfer(B, n_pos, g.R, g.cosT, g.sinT, g.theta, g.v, d_K, d_H, tws, tws_bytes, chunk, s, sel);
}

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct PropPlan {        // workspace plan of wpccc_propagate
    bool two; int n_groups, n_units, W; size_t fixed, per_idx_single, per_idx_double, tws;
};

PropPlan plan_propagate(const wpccc_basis *B, int n_traj, int n_groups, int n_units) {
    PropPlan P{};
    P.two = B->n_centres == 2; P.n_groups = n_groups; P.n_units = n_units;
    const size_t N = B->n_tot;
    if (P.two) {
        const size_t NT = B->c[0].n_states, NP = B->c[1].n_states;
        P.tws = align256(wp_transfer_ws_bytes(B, wp_transfer_default_chunk(B)));
        P.fixed = P.tws + 64 * 1024 + (size_t)n_traj * 64;
        P.per_idx_single = (size_t)n_traj * (6 * 8 + (size_t)B->E_tot * 8) + 4096;                                   // geometry + F
        P.per_idx_double = (size_t)n_traj * (N * N * 16 + NP * NT * 16 + NP * NP * 16) + 4096;                       // H0, K, Ainv
    } else {
        P.tws = 0;
        P.fixed = 64 * 1024 + (size_t)n_traj * 64 + (size_t)n_units * sizeof(SweepUnit);
        P.per_idx_single = (size_t)n_groups * (6 * 8 + (size_t)B->E_tot * 8) + 4096;
        P.per_idx_double = (size_t)n_groups * N * (size_t)wp_sweep1_ld((int)N) * 8 + 4096;                                      // real D^T (even row stride)
    }
    return P;
}
size_t plan_bytes(const PropPlan &P, int W) { const size_t n_idx = 2 * (size_t)W + 1; return P.fixed + n_idx * (P.per_idx_single + 2 * P.per_idx_double) + 16384; }

}  // namespace

extern "C" size_t wpccc_workspace_bytes(const wpccc_basis *B, int n_traj, int n_steps, int what) {
    if (!B || n_traj < 1) return 0;
    if (what == 0) {
        const size_t N = B->n_tot;
        size_t per = 9 * 8 + (size_t)B->E_tot * 8 + 64 + N * N * 16;           // the terms wpccc_matrix_elements checks (H scratch when no H output)
        if (B->n_centres == 2) per += (size_t)B->c[0].n_states * B->c[1].n_states * 16;
        size_t tot = per * (size_t)n_traj + 65536;
        if (B->n_centres == 2) tot += align256(wp_transfer_ws_bytes(B, std::min(n_traj, wp_transfer_default_chunk(B))));
        return tot;
    }
    // propagate: n_groups <= n_traj (worst case every b distinct)
    PropPlan P = plan_propagate(B, n_traj, n_traj, n_traj);
    if (what == 2) return plan_bytes(P, 1);
    int W = std::max(1, std::min(n_steps, 64));
    while (W > 1 && plan_bytes(P, W) > ((size_t)48 << 30)) W = W / 2;
    size_t tot = plan_bytes(P, W);
    if (P.two && W == std::min(std::max(n_steps, 1), 64) && wp_transfer_mirror_ok(B))     // mirror stash, at most 32 GB
        tot += std::min((size_t)n_traj * (size_t)std::max(n_steps, 1) * wp_transfer_stash_doubles(B) * 8, (size_t)32 << 30) + 4096;
    return tot;
}

extern "C" int wpccc_matrix_elements(const wpccc_basis *Bc, int n_pos, const double *b, const double *z, const double *v, int flags,
                                     double *dS, double *dH, double *dF, void *ws, size_t ws_bytes, void *stream) {
    if (!Bc) WP_FAIL(WPCCC_EINVAL, "basis is NULL");
    wpccc_basis *B = const_cast<wpccc_basis *>(Bc);
    if (n_pos < 0 || (n_pos > 0 && (!b || !z || !v))) WP_FAIL(WPCCC_EINVAL, "n_pos < 0 or position arrays NULL");
    if (n_pos == 0) return 0;
    if (!ws) WP_FAIL(WPCCC_ENOMEM, "workspace is NULL");
    for (int p = 0; p < n_pos; ++p) {
        if (!(v[p] > 0.0)) WP_FAIL(WPCCC_EINVAL, "v[%d] must be > 0", p);
        if (!(b[p] >= 0.0) || !(b[p] * b[p] + z[p] * z[p] > 0.0)) WP_FAIL(WPCCC_EINVAL, "position %d: need b >= 0 and R > 0", p);
    }
    cudaStream_t s = (cudaStream_t)stream;
    wp_timing_reset(B);
    B->tab_zeroed = nullptr;
    const bool two = B->n_centres == 2;
    const int NT = B->c[0].n_states, NP = two ? B->c[1].n_states : 0, N = NT + NP;
    // block size from the workspace
    size_t per = 9 * 8 + (size_t)B->E_tot * 8 + 64;
    if (two) per += (size_t)NP * NT * 16 + (dH ? 0 : (size_t)N * N * 16);
    else per += dH ? 0 : (size_t)N * N * 16;
    const int tchunk = two ? wp_transfer_default_chunk(B) : 0;
    const size_t tws_bytes = two ? align256(wp_transfer_ws_bytes(B, std::min(n_pos, tchunk))) : 0;
    if (ws_bytes < tws_bytes + 65536 + per) WP_FAIL(WPCCC_ENOMEM, "workspace too small: need at least %zu bytes", tws_bytes + 65536 + per);
    const int blk = (int)std::min<size_t>((size_t)n_pos, (ws_bytes - tws_bytes - 65536) / per);
    Carver cv(ws, ws_bytes);
    void *tws = two ? cv.take<char>(tws_bytes) : nullptr;
    double *d_b = cv.take<double>(blk), *d_z = cv.take<double>(blk), *d_v = cv.take<double>(blk);
    GeomOut g = carve_geom(cv, blk);
    double *d_F = cv.take<double>((size_t)blk * B->E_tot);
    double *d_K = two ? cv.take<double>((size_t)blk * NP * NT * 2) : nullptr;
    double *d_Htmp = dH ? nullptr : cv.take<double>((size_t)blk * N * N * 2);
    if (!cv.ok) WP_FAIL(WPCCC_ENOMEM, "workspace too small");
    for (int p0 = 0; p0 < n_pos; p0 += blk) {
        const int np = std::min(blk, n_pos - p0);
        WP_CUDA(cudaMemcpyAsync(d_b, b + p0, np * sizeof(double), cudaMemcpyHostToDevice, s));
        WP_CUDA(cudaMemcpyAsync(d_z, z + p0, np * sizeof(double), cudaMemcpyHostToDevice, s));
        WP_CUDA(cudaMemcpyAsync(d_v, v + p0, np * sizeof(double), cudaMemcpyHostToDevice, s));
        wp_span_begin(B, FAM_OTHER, s);
        k_geometry_list<<<(np + 127) / 128, 128, 0, s>>>(np, d_b, d_z, d_v, g);
        wp_span_end(B, s, 1);
        double *H = dH ? dH + (size_t)p0 * N * N * 2 : d_Htmp;
        int rc;
        if (two) {
            WP_CUDA(cudaMemsetAsync(H, 0, (size_t)np * N * N * 16, s));
            rc = elements_two_centre(B, np, g, d_F, d_K, H, tws, tws_bytes, tchunk, s);
        } else {
            rc = wp_direct_gemm(B, np, g.R, d_F, B->E_tot, s);
            if (!rc) rc = wp_direct_assemble(B, 0, np, g.cosT, d_F, B->E_tot, H, N, (long long)N * N, 1, s);
        }
        if (rc) return rc;
        if (dF) WP_CUDA(cudaMemcpyAsync(dF + (size_t)p0 * B->E_tot, d_F, (size_t)np * B->E_tot * 8, cudaMemcpyDeviceToDevice, s));
        if (dS || (dH && (flags & 1))) {
            ComposeArgs ca{};
            ca.K = d_K; ca.S = dS ? dS + (size_t)p0 * N * N * 2 : nullptr; ca.H = (dH && (flags & 1)) ? H : nullptr; ca.z = g.z; ca.v = g.v;
            ca.st_rad_T = B->c[0].d_st_rad; ca.eps_T = B->c[0].d_eps;
            ca.st_rad_P = two ? B->c[1].d_st_rad : nullptr; ca.eps_P = two ? B->c[1].d_eps : nullptr;
            ca.NT = NT; ca.NP = NP; ca.phases = flags & 1;
            dim3 grid(np, std::min(64, (N * N + 255) / 256));
            wp_span_begin(B, FAM_OTHER, s);
            k_compose<<<grid, 256, 0, s>>>(ca);
            wp_span_end(B, s, 1);
        }
        WP_CUDA(cudaGetLastError());
        if (p0 + blk < n_pos) WP_CUDA(cudaStreamSynchronize(s));    // the staging buffers are reused by the next block
    }
    return 0;
}

extern "C" int wpccc_propagate(const wpccc_basis *Bc, int n_traj, const double *b, const double *v, double z_min, double z_max,
                               int n_steps, int init_state, double *dC, double *d_norm_drift, void *ws, size_t ws_bytes, void *stream) {
    if (!Bc) WP_FAIL(WPCCC_EINVAL, "basis is NULL");
    wpccc_basis *B = const_cast<wpccc_basis *>(Bc);
    if (n_traj < 0 || n_steps < 1 || !(z_max > z_min)) WP_FAIL(WPCCC_EINVAL, "need n_traj >= 0, n_steps >= 1, z_max > z_min");
    if (n_traj == 0) return 0;
    if (!b || !v || !dC) WP_FAIL(WPCCC_EINVAL, "b, v or dC is NULL");
    const int N = B->n_tot;
    if (init_state < 0 || init_state >= N) WP_FAIL(WPCCC_EINVAL, "init_state out of range");
    for (int t = 0; t < n_traj; ++t) if (!(b[t] > 0.0) || !(v[t] > 0.0)) WP_FAIL(WPCCC_EINVAL, "trajectory %d: need b > 0 and v > 0", t);
    if (!ws) WP_FAIL(WPCCC_ENOMEM, "workspace is NULL");
    cudaStream_t s = (cudaStream_t)stream, e = B->side, sw = B->hi;
    wp_timing_reset(B);
    B->tab_zeroed = nullptr;
    const bool two = B->n_centres == 2;
    const double h = (z_max - z_min) / n_steps;

    // one-centre: trajectories with the same b share every matrix (D^T depends on (b, z) only)
    std::vector<double> ub; std::vector<int> group_of(n_traj);
    std::vector<SweepUnit> units;
    int nv = 1, rows_per_chunk = 1, ring_stages = 2;
    const int ldD = wp_sweep1_ld(N);
    if (!two) {
        std::map<double, int> idx;
        std::vector<std::vector<int>> members;
        for (int t = 0; t < n_traj; ++t) {
            auto it = idx.find(b[t]);
            if (it == idx.end()) { it = idx.emplace(b[t], (int)ub.size()).first; ub.push_back(b[t]); members.emplace_back(); }
            group_of[t] = it->second; members[it->second].push_back(t);
        }
        // units of up to nv trajectories; nv limited by the sweep kernel's shared memory
        wp_sweep1_plan(N, B->c[0].n_rad, &nv, &rows_per_chunk, &ring_stages);
        for (size_t g = 0; g < members.size(); ++g)
            for (size_t k = 0; k < members[g].size(); k += nv) {
                SweepUnit u{}; u.group = (int)g; u.n = (int)std::min<size_t>(nv, members[g].size() - k);
                for (int q = 0; q < u.n; ++q) u.traj[q] = members[g][k + q];
                units.push_back(u);
            }
    }
    const int n_groups = two ? n_traj : (int)ub.size();
    PropPlan P = plan_propagate(B, n_traj, n_groups, (int)units.size());
    if (ws_bytes < plan_bytes(P, 1)) WP_FAIL(WPCCC_ENOMEM, "workspace too small: need at least %zu bytes", plan_bytes(P, 1));
    int W = std::min(n_steps, 64);
    while (W > 1 && plan_bytes(P, W) > ws_bytes) --W;
    const int n_idx_max = 2 * W + 1;

    Carver cv(ws, ws_bytes);
    double *d_b = cv.take<double>(n_groups), *d_v = cv.take<double>(n_traj);
    SweepUnit *d_units = two ? nullptr : cv.take<SweepUnit>(units.size());
    void *tws = two ? cv.take<char>(P.tws) : nullptr;
    const size_t npos_max = (size_t)n_groups * n_idx_max;
    GeomOut g = carve_geom(cv, npos_max);
    double *d_F = cv.take<double>(npos_max * B->E_tot);
    double *d_H[2] = {nullptr, nullptr}, *d_K[2] = {nullptr, nullptr}, *d_LU[2] = {nullptr, nullptr}, *d_D[2] = {nullptr, nullptr};
    const size_t NT = B->c[0].n_states, NP = two ? B->c[1].n_states : 0;
    for (int k = 0; k < 2; ++k) {
        if (two) {
            d_H[k] = cv.take<double>(npos_max * N * N * 2); d_K[k] = cv.take<double>(npos_max * NP * NT * 2);
            d_LU[k] = cv.take<double>(npos_max * NP * NP * 2);
        } else d_D[k] = cv.take<double>(npos_max * N * ldD);
    }
    if (!cv.ok) WP_FAIL(WPCCC_ENOMEM, "workspace too small (internal plan mismatch)");
    // Mirror stash: on a z-grid symmetric about 0 the body-frame two-centre integrals at (b, +z) are written by the
    // launch that evaluates (b, -z) (TransferSel, common.cuh); whatever the workspace has left beyond the window
    // buffers holds the n_st half-step positions per trajectory that follow z = 0.
    TransferSel sel{}; bool mirror = false;
    if (two && std::fabs(z_min + z_max) <= 1e-14 * std::fabs(z_max) && wp_transfer_mirror_ok(B) && !getenv("WPCCC_NO_MIRROR")) {
        const size_t slot = wp_transfer_stash_doubles(B) * 8, left = ws_bytes > cv.off + 4096 ? ws_bytes - cv.off - 4096 : 0;
        const size_t n_st = std::min<size_t>((size_t)n_steps, left / ((size_t)n_traj * slot));
        if (n_st > 0) {
            sel.stash = cv.take<double>((size_t)n_traj * n_st * (slot / 8));
            sel.n_st = (int)n_st; sel.n_groups = n_traj; sel.i_mid = n_steps; mirror = cv.ok;
        }
    }

    if (two) WP_CUDA(cudaMemcpyAsync(d_b, b, n_traj * sizeof(double), cudaMemcpyHostToDevice, s));
    else WP_CUDA(cudaMemcpyAsync(d_b, ub.data(), ub.size() * sizeof(double), cudaMemcpyHostToDevice, s));
    WP_CUDA(cudaMemcpyAsync(d_v, v, n_traj * sizeof(double), cudaMemcpyHostToDevice, s));
    if (!two) WP_CUDA(cudaMemcpyAsync(d_units, units.data(), units.size() * sizeof(SweepUnit), cudaMemcpyHostToDevice, s));
    WP_CUDA(cudaMemsetAsync(B->d_status, 0, 4 * sizeof(int), s));
    k_init_amplitudes<<<(unsigned)(((size_t)n_traj * N + 255) / 256), 256, 0, s>>>(dC, n_traj, N, init_state);
    if (d_norm_drift) WP_CUDA(cudaMemsetAsync(d_norm_drift, 0, n_traj * sizeof(double), s));
    const int tchunk = two ? wp_transfer_default_chunk(B) : 0;

    // element stream `e` and sweep stream `sw` fork from the caller's stream and join back at the end
    cudaEvent_t ev_elem[2], ev_sweep[2];
    for (int k = 0; k < 2; ++k) { WP_CUDA(cudaEventCreateWithFlags(&ev_elem[k], cudaEventDisableTiming)); WP_CUDA(cudaEventCreateWithFlags(&ev_sweep[k], cudaEventDisableTiming)); }
    WP_CUDA(cudaEventRecord(B->ev_fork, s));
    WP_CUDA(cudaStreamWaitEvent(e, B->ev_fork, 0));
    WP_CUDA(cudaStreamWaitEvent(sw, B->ev_fork, 0));
    int rc = 0, wi = 0;
    for (int s0 = 0; s0 < n_steps && !rc; s0 += W, ++wi) {
        const int steps = std::min(W, n_steps - s0), n_idx = 2 * steps + 1, buf = wi & 1;
        const long long i0 = 2LL * s0;
        const int n_pos = n_groups * n_idx;
        if (wi >= 2) WP_CUDA(cudaStreamWaitEvent(e, ev_sweep[buf], 0));     // buffer `buf` free again
        wp_span_begin(B, FAM_OTHER, e);
        k_geometry_grid<<<(n_pos + 127) / 128, 128, 0, e>>>(n_groups, n_idx, d_b, two ? d_v : nullptr, i0, z_min, h, g);
        wp_span_end(B, e, 1);
        if (two) {
            // no clearing of d_H[buf]: the assembly kernels write every element of D^T, D^P and the rotation kernel every
            // element of H_PT, H_TP at every position of the window (evaluated or fetched from the mirror stash)
            if (mirror) {
                sel.n_idx = n_idx; sel.i0 = i0;
                sel.n_pre = (int)std::max<long long>(0, std::min<long long>(n_idx, sel.i_mid + 1 - i0));
                sel.suf0 = (int)std::max<long long>(sel.n_pre, std::min<long long>(n_idx, sel.i_mid + sel.n_st + 1 - i0));
            }
            rc = elements_two_centre(B, n_pos, g, d_F, d_K[buf], d_H[buf], tws, P.tws, tchunk, e, mirror ? &sel : nullptr);
            if (!rc) rc = wp_factor(B, n_pos, d_K[buf], d_LU[buf], e);
        } else {
            rc = wp_direct_gemm(B, n_pos, g.R, d_F, B->E_tot, e);
            if (!rc) rc = wp_direct_assemble(B, 0, n_pos, g.cosT, d_F, B->E_tot, d_D[buf], ldD, (long long)N * ldD, 0, e);
        }
        if (rc) break;
        WP_CUDA(cudaEventRecord(ev_elem[buf], e));
        WP_CUDA(cudaStreamWaitEvent(sw, ev_elem[buf], 0));
        if (two) {
            Sweep2Args a{};
            a.H = d_H[buf]; a.K = d_K[buf]; a.Ainv = d_LU[buf];
            a.st_rad_T = B->c[0].d_st_rad; a.st_rad_P = B->c[1].d_st_rad; a.eps_T = B->c[0].d_eps; a.eps_P = B->c[1].d_eps;
            a.v = d_v; a.C = dC; a.drift = d_norm_drift; a.NT = (int)NT; a.NP = (int)NP; a.n_idx = n_idx; a.steps = steps; a.i0 = i0; a.z_min = z_min; a.h = h;
            rc = wp_sweep_two_centre(B, n_traj, a, sw);
        } else {
            Sweep1Args a{};
            a.units = d_units; a.D = d_D[buf]; a.st_rad = B->c[0].d_st_rad; a.eps = B->c[0].d_eps; a.v = d_v; a.C = dC; a.drift = d_norm_drift;
            a.N = N; a.n_rad = B->c[0].n_rad; a.n_idx = n_idx; a.ldD = ldD; a.nv = nv; a.rows_per_chunk = rows_per_chunk; a.ring_stages = ring_stages; a.steps = steps; a.i0 = i0; a.z_min = z_min; a.h = h;
            rc = wp_sweep_one_centre(B, (int)units.size(), a, sw);
        }
        if (rc) break;
        WP_CUDA(cudaEventRecord(ev_sweep[buf], sw));
    }
    // join: the caller's stream waits for everything enqueued on the element stream
    cudaEventRecord(B->ev_join, e);
    cudaStreamWaitEvent(s, B->ev_join, 0);
    cudaEventRecord(B->ev_join2, sw);
    cudaStreamWaitEvent(s, B->ev_join2, 0);
    int status[4] = {0, 0, 0, 0};
    cudaError_t ce = cudaMemcpyAsync(status, B->d_status, sizeof status, cudaMemcpyDeviceToHost, s);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(s);
    cudaStreamSynchronize(e);
    cudaStreamSynchronize(sw);
    for (int k = 0; k < 2; ++k) { cudaEventDestroy(ev_elem[k]); cudaEventDestroy(ev_sweep[k]); }
    if (rc) return rc;
    if (ce != cudaSuccess) WP_FAIL(WPCCC_ECUDA, "propagate: %s", cudaGetErrorString(ce));
    if (status[0] == 1) WP_FAIL(WPCCC_ESINGULAR, "zero pivot in the overlap factorisation (window-local position %d)", status[1] - 1);
    if (status[0] == 2) WP_FAIL(WPCCC_ESINGULAR, "|S_PT| >= 1 at window-local position %d: pivot-order precondition violated", status[1] - 1);
    return 0;
}

extern "C" int wpccc_probabilities(const wpccc_basis *B, int n_traj, const double *dC, const double *b, const int *vgroup, int n_vgroups,
                                   int init_state, double *P_state, double *P_nl, double *P_class, double *sigma_nl, double *sigma_class,
                                   void *stream) {
    if (!B || !dC || n_traj < 1) WP_FAIL(WPCCC_EINVAL, "basis/dC NULL or n_traj < 1");
    const int N = B->n_tot;
    if (init_state < 0 || init_state >= N) WP_FAIL(WPCCC_EINVAL, "init_state out of range");
    if ((sigma_nl || sigma_class) && (!b || !vgroup || n_vgroups < 1)) WP_FAIL(WPCCC_EINVAL, "cross sections need b, vgroup, n_vgroups");
    if (sigma_nl && !P_nl) WP_FAIL(WPCCC_EINVAL, "sigma_nl needs P_nl");
    if (sigma_class && !P_class) WP_FAIL(WPCCC_EINVAL, "sigma_class needs P_class");
    cudaStream_t s = (cudaStream_t)stream;
    int n_rad_tot = 0;
    std::vector<int> st_rad_glob, rad_class;
    for (int c = 0; c < B->n_centres; ++c) {
        for (int j = 0; j < B->c[c].n_states; ++j) st_rad_glob.push_back(n_rad_tot + B->c[c].st_rad[j]);
        n_rad_tot += B->c[c].n_rad;
    }
    const int r_init = st_rad_glob[init_state];
    for (int c = 0, r = 0; c < B->n_centres; ++c)
        for (int a = 0; a < B->c[c].n_rad; ++a, ++r)
            rad_class.push_back(r == r_init ? 0 : (c == 0 ? (B->c[c].kind[a] == 0 ? 1 : 2) : (B->c[c].kind[a] == 0 ? 3 : 4)));
    // small index tables: temporary device buffers (index marshalling, freed on return)
    int *d_idx = nullptr;
    const size_t n_int = (size_t)N + n_rad_tot + n_traj + n_vgroups + 1;
    WP_CUDA(cudaMallocAsync(&d_idx, n_int * sizeof(int) + (size_t)n_traj * sizeof(double) + 64, s));
    int *d_srg = d_idx, *d_cls = d_idx + N, *d_order = d_cls + n_rad_tot, *d_goff = d_order + n_traj;
    double *d_bb = reinterpret_cast<double *>(((uintptr_t)(d_goff + n_vgroups + 1) + 15) & ~(uintptr_t)15);
    WP_CUDA(cudaMemcpyAsync(d_srg, st_rad_glob.data(), N * sizeof(int), cudaMemcpyHostToDevice, s));
    WP_CUDA(cudaMemcpyAsync(d_cls, rad_class.data(), n_rad_tot * sizeof(int), cudaMemcpyHostToDevice, s));
    ProbArgs a{};
    a.C = dC; a.n_traj = n_traj; a.N = N; a.n_rad_tot = n_rad_tot; a.st_rad_glob = d_srg; a.rad_class = d_cls;
    a.P_state = P_state; a.P_nl = P_nl; a.P_class = P_class;
    k_probabilities<<<n_traj, 128, n_rad_tot * sizeof(double), s>>>(a);
    std::vector<int> order, goff;
    if (sigma_nl || sigma_class) {
        for (int g = 0; g < n_vgroups; ++g) {
            goff.push_back((int)order.size());
            std::vector<int> m;
            for (int t = 0; t < n_traj; ++t) if (vgroup[t] == g) m.push_back(t);
            std::stable_sort(m.begin(), m.end(), [&](int x, int y) { return b[x] < b[y]; });
            order.insert(order.end(), m.begin(), m.end());
        }
        goff.push_back((int)order.size());
        order.resize(n_traj, 0);
        WP_CUDA(cudaMemcpyAsync(d_order, order.data(), n_traj * sizeof(int), cudaMemcpyHostToDevice, s));
        WP_CUDA(cudaMemcpyAsync(d_goff, goff.data(), goff.size() * sizeof(int), cudaMemcpyHostToDevice, s));
        WP_CUDA(cudaMemcpyAsync(d_bb, b, n_traj * sizeof(double), cudaMemcpyHostToDevice, s));
        if (sigma_nl) k_cross_sections<<<n_vgroups, 128, 0, s>>>(P_nl, n_rad_tot, d_bb, d_order, d_goff, sigma_nl);
        if (sigma_class) k_cross_sections<<<n_vgroups, 32, 0, s>>>(P_class, 5, d_bb, d_order, d_goff, sigma_class);
    }
    WP_CUDA(cudaGetLastError());
    WP_CUDA(cudaStreamSynchronize(s));     // host index vectors must outlive the copies
    WP_CUDA(cudaFreeAsync(d_idx, s));
    return 0;
}

// ---------------------------------------------------------------------------------------------- FP64 peak probe
namespace {
__global__ void __launch_bounds__(256) k_peak_dfma(double *out, int iters, double x) {
    double a[16];
    #pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = threadIdx.x * 1e-3 + i;
    const double m = 1.0 + x, c = x;
    for (int it = 0; it < iters; ++it) {
        #pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fma(a[i], m, c);
    }
    double s = 0.0;
    #pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == 12345.678) out[0] = s;
}
__global__ void __launch_bounds__(256) k_peak_dmma(double *out, int iters, double x) {
    double c[8][2];
    #pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x * 1e-3; c[i][1] = i; }
    double a = 1.0 + x * threadIdx.x, b = x;
    for (int it = 0; it < iters; ++it) {
        #pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
    #pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[0] = s;
}
}  // namespace

extern "C" double wpccc_fp64_peak(int kind, void *stream) {
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        wp_set_error("no CUDA device"); return (double)WPCCC_ECUDA;
    }
    double *d = nullptr;
    if (cudaMalloc(&d, 64) != cudaSuccess) { wp_set_error("cudaMalloc failed"); return (double)WPCCC_ECUDA; }
    const int iters = 20000, blocks = sms * 8;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, s);
        if (kind == 0) k_peak_dfma<<<blocks, 256, 0, s>>>(d, iters, 1e-9);
        else k_peak_dmma<<<blocks, 256, 0, s>>>(d, iters, 1e-9);
        cudaEventRecord(e1, s);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = (double)WPCCC_ECUDA; break; }
        float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
        // DFMA: 16 FMA per thread per iteration; DMMA: 8 mma per warp per iteration, 8*8*4 FMA each
        const double flops = (kind == 0) ? 2.0 * 16 * iters * 256.0 * blocks : 2.0 * 8 * 256.0 * iters * 8.0 * blocks;
        if (rep > 0) best = std::max(best, flops / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    return best;
}
