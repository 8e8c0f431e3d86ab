// a7 factorisation and a8 RK4 sweep (Algorithm 1; eq. (2)-(5), L49-65).
//
// The matrices do not depend on the amplitudes, so they are produced for a whole window of steps by the element
// kernels; only the sweep below is sequential in z.  Matrices are stored WITHOUT the interaction-picture phases
// (A2): with P = diag(e^{i eps z/v}), S = P S0 P^H and H = P H0 P^H, hence
//     dc/dz = -(i/v) S^{-1} H c = -(i/v) P S0^{-1} H0 P^H c,
// i.e. rotate the stage vector by P^H, multiply/solve with the phase-free matrices, rotate back by P.
//
// a7: S0 = [[I, K^H], [K, I]].  Gaussian elimination with partial pivoting of S0 picks the unit diagonal as pivot
// in its first N_T columns whenever every |K_ij| < 1 (the other candidates in column j are exactly K[:,j]), which
// leaves the Schur complement A = I - K K^H in the projectile block.  The kernel forms A, checks |K_ij| < 1, and
// continues the same elimination (partial pivoting, first maximal pivot wins) on A.  Solve:
//     y_P' = y_P - K y_T;  A w_P = y_P';  w_T = y_T - K^H w_P.
#include "sweep.cuh"

namespace {

struct cplx { double x, y; };
__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x}; }
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) { return {a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y}; }  // a * conj(b)
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return {a.x + b.x, a.y + b.y}; }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return {a.x - b.x, a.y - b.y}; }
__device__ __forceinline__ double warp_sum(double v) {
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double zpos(double z_min, double h, long long i) { return __dadd_rn(z_min, __dmul_rn(0.5 * (double)i, h)); }

// ------------------------------------------------------------------ one-centre sweep
// grid = units; block = 256.  Dynamic smem: C, A, X, Knew [nv][N] complex, ph [nv][n_rad] complex, red[8].
__global__ void __launch_bounds__(256) k_sweep1(const Sweep1Args a) {
    extern __shared__ __align__(16) double sm[];
    const SweepUnit u = a.units[blockIdx.x];
    const int N = a.N, nv = u.n, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
    cplx *C = reinterpret_cast<cplx *>(sm);
    cplx *Acc = C + SWEEP_NV * N;
    cplx *X = Acc + SWEEP_NV * N;
    cplx *Kn = X + SWEEP_NV * N;
    cplx *ph = Kn + SWEEP_NV * N;               // [nv][n_rad]
    __shared__ double red[SWEEP_NV][8];
    double vel[SWEEP_NV];
    for (int q = 0; q < SWEEP_NV; ++q) vel[q] = (q < nv) ? a.v[u.traj[q]] : 1.0;

    for (int q = 0; q < nv; ++q)
        for (int j = tid; j < N; j += blockDim.x) {
            const double *src = a.C + ((size_t)u.traj[q] * N + j) * 2;
            C[q * N + j] = {src[0], src[1]};
        }
    double drift[SWEEP_NV];
    for (int q = 0; q < SWEEP_NV; ++q) drift[q] = (a.drift && q < nv) ? a.drift[u.traj[q]] : 0.0;
    __syncthreads();

    const double h = a.h;
    for (int s = 0; s < a.steps; ++s) {
        for (int j = tid; j < nv * N; j += blockDim.x) { Acc[j] = {0.0, 0.0}; Kn[j] = {0.0, 0.0}; }
        __syncthreads();
        #pragma unroll 1
        for (int st = 0; st < 4; ++st) {
            const int li = 2 * s + (st == 0 ? 0 : (st == 3 ? 2 : 1));       // local half-step index of this stage
            const double alpha = (st == 0) ? 0.0 : (st == 3 ? h : 0.5 * h);
            const double wgt = (st == 0 || st == 3) ? 1.0 : 2.0;
            const double z = zpos(a.z_min, h, a.i0 + li);
            for (int j = tid; j < nv * a.n_rad; j += blockDim.x) {
                int q = j / a.n_rad, r = j % a.n_rad;
                double sn, cs; sincos(a.eps[r] * z / vel[q], &sn, &cs);
                ph[j] = {cs, sn};
            }
            __syncthreads();
            // X = P^H (C + alpha * Kn)
            for (int j = tid; j < nv * N; j += blockDim.x) {
                int q = j / N, col = j % N;
                cplx x = {C[j].x + alpha * Kn[j].x, C[j].y + alpha * Kn[j].y};
                X[j] = cmulc(x, ph[q * a.n_rad + a.st_rad[col]]);
            }
            __syncthreads();
            const double *D = a.D + ((size_t)u.group * a.n_idx + li) * (size_t)N * N;
            for (int row = warp; row < N; row += nw) {
                const double *Dr = D + (size_t)row * N;
                double sr[SWEEP_NV], si[SWEEP_NV];
                #pragma unroll
                for (int q = 0; q < SWEEP_NV; ++q) { sr[q] = 0.0; si[q] = 0.0; }
                for (int col = lane; col < N; col += 32) {
                    const double d = Dr[col];
                    #pragma unroll
                    for (int q = 0; q < SWEEP_NV; ++q) if (q < nv) { cplx x = X[q * N + col]; sr[q] += d * x.x; si[q] += d * x.y; }
                }
                #pragma unroll
                for (int q = 0; q < SWEEP_NV; ++q) if (q < nv) {
                    double yr = warp_sum(sr[q]), yi = warp_sum(si[q]);
                    if (lane == 0) {
                        // k = -(i/v) P y
                        cplx y = cmul({yr, yi}, ph[q * a.n_rad + a.st_rad[row]]);
                        cplx k = {y.y / vel[q], -y.x / vel[q]};
                        Kn[q * N + row] = k;
                        Acc[q * N + row].x += wgt * k.x; Acc[q * N + row].y += wgt * k.y;
                    }
                }
            }
            __syncthreads();
        }
        for (int j = tid; j < nv * N; j += blockDim.x) { C[j].x += (h / 6.0) * Acc[j].x; C[j].y += (h / 6.0) * Acc[j].y; }
        __syncthreads();
        if (a.drift) {
            for (int q = 0; q < nv; ++q) {
                double part = 0.0;
                for (int j = tid; j < N; j += blockDim.x) part += C[q * N + j].x * C[q * N + j].x + C[q * N + j].y * C[q * N + j].y;
                part = warp_sum(part);
                if (lane == 0) red[q][warp] = part;
            }
            __syncthreads();
            for (int q = 0; q < nv; ++q) {
                double tot = 0.0;
                for (int w = 0; w < nw; ++w) tot += red[q][w];
                drift[q] = fmax(drift[q], fabs(tot - 1.0));
            }
            __syncthreads();
        }
    }
    for (int q = 0; q < nv; ++q) {
        for (int j = tid; j < N; j += blockDim.x) {
            double *dst = a.C + ((size_t)u.traj[q] * N + j) * 2;
            dst[0] = C[q * N + j].x; dst[1] = C[q * N + j].y;
        }
        if (a.drift && tid == 0) a.drift[u.traj[q]] = drift[q];
    }
}

// ------------------------------------------------------------------ a7: Schur complement + LU
// grid = positions; block = 256.  A (column-major, ld = NP) lives in shared memory when it fits, else in LU (global).
struct FactorArgs { const double *K; double *LU; int *piv; int *status; int NT, NP, use_smem; };

__global__ void __launch_bounds__(256) k_factor(const FactorArgs a) {
    extern __shared__ __align__(16) double sm[];
    const int NP = a.NP, NT = a.NT, tid = threadIdx.x, nt = blockDim.x;
    const size_t p = blockIdx.x;
    const cplx *K = reinterpret_cast<const cplx *>(a.K) + p * (size_t)NP * NT;
    cplx *G = reinterpret_cast<cplx *>(a.LU) + p * (size_t)NP * NP;
    cplx *A = a.use_smem ? reinterpret_cast<cplx *>(sm) : G;
    int *piv = a.piv + p * NP;
    __shared__ double s_red[256]; __shared__ int s_idx[256]; __shared__ int s_flag;
    if (tid == 0) s_flag = 0;
    __syncthreads();
    // |K_ij| < 1 check (pivot-order precondition)
    int bad = 0;
    for (int i = tid; i < NP * NT; i += nt) { cplx k = K[i]; if (!(k.x * k.x + k.y * k.y < 1.0)) bad = 1; }
    if (bad) s_flag = 2;
    // A[r][s] = delta_rs - sum_i K[r][i] conj(K[s][i]), accumulated in the order i = 0..NT-1 (the elimination order)
    for (int e = tid; e < NP * NP; e += nt) {
        const int r = e % NP, s = e / NP;
        const cplx *Kr = K + (size_t)r * NT, *Ks = K + (size_t)s * NT;
        double ar = (r == s) ? 1.0 : 0.0, ai = 0.0;
        for (int i = 0; i < NT; ++i) { cplx x = Kr[i], y = Ks[i]; ar -= x.x * y.x + x.y * y.y; ai -= x.y * y.x - x.x * y.y; }
        A[(size_t)s * NP + r] = {ar, ai};
    }
    __syncthreads();
    for (int j = 0; j < NP; ++j) {
        // pivot search in column j, rows j..NP-1 (first maximal |.| wins)
        double best = -1.0; int bi = j;
        for (int i = j + tid; i < NP; i += nt) { cplx x = A[(size_t)j * NP + i]; double m = x.x * x.x + x.y * x.y; if (m > best) { best = m; bi = i; } }
        s_red[tid] = best; s_idx[tid] = bi;
        __syncthreads();
        for (int o = nt >> 1; o > 0; o >>= 1) {
            if (tid < o) {
                double m2 = s_red[tid + o]; int i2 = s_idx[tid + o];
                if (m2 > s_red[tid] || (m2 == s_red[tid] && i2 < s_idx[tid])) { s_red[tid] = m2; s_idx[tid] = i2; }
            }
            __syncthreads();
        }
        const int pr = s_idx[0];
        const double pm = s_red[0];
        if (tid == 0) { piv[j] = pr; if (!(pm > 0.0)) s_flag = 1; }
        if (pr != j)
            for (int c = tid; c < NP; c += nt) { cplx t = A[(size_t)c * NP + j]; A[(size_t)c * NP + j] = A[(size_t)c * NP + pr]; A[(size_t)c * NP + pr] = t; }
        __syncthreads();
        const cplx d = A[(size_t)j * NP + j];
        const double dn = d.x * d.x + d.y * d.y;
        const cplx dinv = (dn > 0.0) ? cplx{d.x / dn, -d.y / dn} : cplx{0.0, 0.0};
        __syncthreads();
        for (int i = j + 1 + tid; i < NP; i += nt) A[(size_t)j * NP + i] = cmul(A[(size_t)j * NP + i], dinv);
        __syncthreads();
        // trailing update A[i][c] -= L[i][j] * U[j][c], i, c > j
        const int rem = NP - 1 - j;
        for (int e = tid; e < rem * rem; e += nt) {
            const int i = j + 1 + e % rem, c = j + 1 + e / rem;
            A[(size_t)c * NP + i] = csub(A[(size_t)c * NP + i], cmul(A[(size_t)j * NP + i], A[(size_t)c * NP + j]));
        }
        __syncthreads();
    }
    if (a.use_smem) for (int e = tid; e < NP * NP; e += nt) G[e] = A[e];
    if (tid == 0 && s_flag) { atomicMax(a.status, s_flag); atomicCAS(a.status + 1, 0, (int)p + 1); }
}

// ------------------------------------------------------------------ two-centre sweep
// grid = trajectories; block = 256.  smem: C, Acc, X, Kn, Y, W [N] complex + ph [N] complex + partial[8][NT].
__global__ void __launch_bounds__(256) k_sweep2(const Sweep2Args a) {
    extern __shared__ __align__(16) double sm[];
    const int NT = a.NT, NP = a.NP, N = NT + NP, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
    const int t = blockIdx.x;
    cplx *C = reinterpret_cast<cplx *>(sm);
    cplx *Acc = C + N, *X = Acc + N, *Kn = X + N, *Y = Kn + N, *ph = Y + N, *part = ph + N;   // part [nw][NT]
    __shared__ double red[8];
    const double vel = a.v[t], h = a.h;
    for (int j = tid; j < N; j += blockDim.x) { const double *src = a.C + ((size_t)t * N + j) * 2; C[j] = {src[0], src[1]}; }
    double drift = a.drift ? a.drift[t] : 0.0;
    __syncthreads();

    for (int s = 0; s < a.steps; ++s) {
        for (int j = tid; j < N; j += blockDim.x) { Acc[j] = {0.0, 0.0}; Kn[j] = {0.0, 0.0}; }
        __syncthreads();
        #pragma unroll 1
        for (int st = 0; st < 5; ++st) {
            // st = 0..3: RK4 stages; st = 4: norm c^H S c at z_new (only when drift is tracked)
            if (st == 4 && !a.drift) break;
            const int li = 2 * s + (st == 0 ? 0 : (st >= 3 ? 2 : 1));
            const double alpha = (st == 0 || st == 4) ? 0.0 : (st == 3 ? h : 0.5 * h);
            const double wgt = (st == 0 || st == 3) ? 1.0 : 2.0;
            const double z = zpos(a.z_min, h, a.i0 + li);
            const size_t pos = (size_t)t * a.n_idx + li;
            for (int j = tid; j < N; j += blockDim.x) {
                double e = (j < NT) ? a.eps_T[a.st_rad_T[j]] : a.eps_P[a.st_rad_P[j - NT]];
                double sn, cs; sincos(e * z / vel, &sn, &cs);
                ph[j] = {cs, sn};
                cplx x = {C[j].x + alpha * Kn[j].x, C[j].y + alpha * Kn[j].y};
                X[j] = cmulc(x, {cs, sn});
            }
            __syncthreads();
            const cplx *Kp = reinterpret_cast<const cplx *>(a.K) + pos * (size_t)NP * NT;
            if (st == 4) {
                // c^H S c = |c|^2 + 2 Re( X_P^H K X_T )
                double acc = 0.0;
                for (int row = warp; row < NP; row += nw) {
                    double sr = 0.0, si = 0.0;
                    for (int col = lane; col < NT; col += 32) { cplx k = Kp[(size_t)row * NT + col], x = X[col]; sr += k.x * x.x - k.y * x.y; si += k.x * x.y + k.y * x.x; }
                    sr = warp_sum(sr); si = warp_sum(si);
                    acc += 2.0 * (X[NT + row].x * sr + X[NT + row].y * si);
                }
                double nrm = 0.0;
                for (int j = lane + 32 * warp; j < N; j += blockDim.x) nrm += X[j].x * X[j].x + X[j].y * X[j].y;
                nrm = warp_sum(nrm);
                if (lane == 0) red[warp] = acc + nrm;
                __syncthreads();
                double tot = 0.0;
                for (int w = 0; w < nw; ++w) tot += red[w];
                drift = fmax(drift, fabs(tot - 1.0));
                __syncthreads();
                break;
            }
            // Y = H0 X
            const cplx *Hp = reinterpret_cast<const cplx *>(a.H) + pos * (size_t)N * N;
            for (int row = warp; row < N; row += nw) {
                const cplx *Hr = Hp + (size_t)row * N;
                double sr = 0.0, si = 0.0;
                for (int col = lane; col < N; col += 32) { cplx hh = Hr[col], x = X[col]; sr += hh.x * x.x - hh.y * x.y; si += hh.x * x.y + hh.y * x.x; }
                sr = warp_sum(sr); si = warp_sum(si);
                if (lane == 0) Y[row] = {sr, si};
            }
            __syncthreads();
            // Y_P -= K Y_T
            for (int row = warp; row < NP; row += nw) {
                double sr = 0.0, si = 0.0;
                for (int col = lane; col < NT; col += 32) { cplx k = Kp[(size_t)row * NT + col], x = Y[col]; sr += k.x * x.x - k.y * x.y; si += k.x * x.y + k.y * x.x; }
                sr = warp_sum(sr); si = warp_sum(si);
                if (lane == 0) { Y[NT + row].x -= sr; Y[NT + row].y -= si; }
            }
            __syncthreads();
            // A w_P = Y_P by the LU factors (column-major), in place in Y_P
            const cplx *LU = reinterpret_cast<const cplx *>(a.LU) + pos * (size_t)NP * NP;
            const int *piv = a.piv + pos * NP;
            cplx *yp = Y + NT;
            if (tid == 0) for (int j = 0; j < NP; ++j) { int pr = piv[j]; if (pr != j) { cplx tt = yp[j]; yp[j] = yp[pr]; yp[pr] = tt; } }
            __syncthreads();
            for (int j = 0; j < NP - 1; ++j) {
                const cplx wj = yp[j];
                __syncthreads();
                for (int i = j + 1 + tid; i < NP; i += blockDim.x) yp[i] = csub(yp[i], cmul(LU[(size_t)j * NP + i], wj));
                __syncthreads();
            }
            for (int j = NP - 1; j >= 0; --j) {
                if (tid == 0) { cplx d = LU[(size_t)j * NP + j]; double dn = d.x * d.x + d.y * d.y; yp[j] = cmul(yp[j], {d.x / dn, -d.y / dn}); }
                __syncthreads();
                const cplx wj = yp[j];
                for (int i = tid; i < j; i += blockDim.x) yp[i] = csub(yp[i], cmul(LU[(size_t)j * NP + i], wj));
                __syncthreads();
            }
            // w_T = Y_T - K^H w_P: partial sums over rows of K per warp, then reduce
            for (int col = lane; col < NT; col += 32) {
                double sr = 0.0, si = 0.0;
                for (int row = warp; row < NP; row += nw) { cplx k = Kp[(size_t)row * NT + col], x = yp[row]; sr += k.x * x.x + k.y * x.y; si += k.x * x.y - k.y * x.x; }
                part[warp * NT + col] = {sr, si};
            }
            __syncthreads();
            for (int col = tid; col < NT; col += blockDim.x) {
                double sr = 0.0, si = 0.0;
                for (int w = 0; w < nw; ++w) { sr += part[w * NT + col].x; si += part[w * NT + col].y; }
                Y[col].x -= sr; Y[col].y -= si;
            }
            __syncthreads();
            // k = -(i/v) P w
            for (int j = tid; j < N; j += blockDim.x) {
                cplx y = cmul(Y[j], ph[j]);
                cplx k = {y.y / vel, -y.x / vel};
                Kn[j] = k; Acc[j].x += wgt * k.x; Acc[j].y += wgt * k.y;
            }
            __syncthreads();
            if (st == 3) {
                for (int j = tid; j < N; j += blockDim.x) { C[j].x += (h / 6.0) * Acc[j].x; C[j].y += (h / 6.0) * Acc[j].y; Kn[j] = {0.0, 0.0}; }
                __syncthreads();
            }
        }
    }
    for (int j = tid; j < N; j += blockDim.x) { double *dst = a.C + ((size_t)t * N + j) * 2; dst[0] = C[j].x; dst[1] = C[j].y; }
    if (a.drift && tid == 0) a.drift[t] = drift;
}

}  // namespace

int wp_sweep_one_centre(wpccc_basis *B, int n_units, const Sweep1Args &a, cudaStream_t s) {
    if (n_units <= 0 || a.steps <= 0) return 0;
    const size_t smem = ((size_t)4 * SWEEP_NV * a.N + (size_t)SWEEP_NV * a.n_rad) * 16;
    if (smem > 220 * 1024) WP_FAIL(WPCCC_EINVAL, "one-centre sweep: N = %d too large for shared memory", a.N);
    WP_CUDA(cudaFuncSetAttribute(k_sweep1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    wp_span_begin(B, FAM_SWEEP, s);
    k_sweep1<<<n_units, 256, smem, s>>>(a);
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}

int wp_sweep_two_centre(wpccc_basis *B, int n_traj, const Sweep2Args &a, cudaStream_t s) {
    if (n_traj <= 0 || a.steps <= 0) return 0;
    const int N = a.NT + a.NP;
    const size_t smem = ((size_t)6 * N + (size_t)8 * a.NT) * 16;
    if (smem > 220 * 1024) WP_FAIL(WPCCC_EINVAL, "two-centre sweep: N = %d too large for shared memory", N);
    WP_CUDA(cudaFuncSetAttribute(k_sweep2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    wp_span_begin(B, FAM_SWEEP, s);
    k_sweep2<<<n_traj, 256, smem, s>>>(a);
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}

int wp_factor(wpccc_basis *B, int n_pos, const double *d_K, double *d_LU, int *d_piv, cudaStream_t s) {
    if (n_pos <= 0) return 0;
    FactorArgs a{};
    a.K = d_K; a.LU = d_LU; a.piv = d_piv; a.status = B->d_status; a.NT = B->c[0].n_states; a.NP = B->c[1].n_states;
    const size_t need = (size_t)a.NP * a.NP * 16;
    a.use_smem = need <= 200 * 1024;
    const size_t smem = a.use_smem ? need : 0;
    WP_CUDA(cudaFuncSetAttribute(k_factor, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 1024)));
    wp_span_begin(B, FAM_FACT, s);
    k_factor<<<n_pos, 256, smem, s>>>(a);
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}
