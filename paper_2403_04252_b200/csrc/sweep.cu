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
// continues the elimination (partial pivoting, first maximal pivot wins) on A in Gauss-Jordan form, which yields
// A^{-1} explicitly: the four solves of an RK4 step then have no sequential dependency chain,
//     y_P' = y_P - K y_T;  w_P = A^{-1} y_P';  w_T = y_T - K^H w_P.
#include <algorithm>
#include <cstdlib>

#include "sweep.cuh"
#include "ptx.cuh"

namespace {

__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, 256;\n" ::: "memory"); }

constexpr int SW_STAGES = 4;
constexpr int SW_CONSUMERS = 256;

constexpr int SW1_CONSUMERS = 224;

// ------------------------------------------------------------------ one-centre sweep
// grid = units (up to NV trajectories that share b, hence D); block = 7 consumer warps + 1 producer warp (256 threads: the full 255 registers per thread).
// The real matrices D(z) do not depend on the amplitudes: the producer warp streams their rows through a
// shared-memory ring with TMA bulk copies (running ahead across stages).  D is symmetric (eq. (6) without the time
// phase), so y_r = sum_c D[c][r] x_c: consumer thread r owns the rows r, r + 224, .. (NTILE of them) of every
// trajectory of the unit, reads element r of each streamed row c (consecutive lanes, conflict-free) and the stage
// vector x_c as a broadcast, and accumulates in registers -- no reductions, no re-reading of x per matrix row.  The
// state (C, RK4 accumulator, phases) of a thread's rows lives in registers; only the stage vector X is shared
// (double-buffered: one block barrier per RK4 stage).  Dynamic smem: ring, then X [2][NV][N] complex.
// NC = 2 (few units, wide basis): a cluster of two CTAs per unit, each streaming one half of the rows of D and multiplying it;
// the partial sums are exchanged through distributed shared memory once per stage (as in k_sweep2).
template <int NTILE, int NV, int NC>
__global__ void __launch_bounds__(SW1_CONSUMERS + 32) k_sweep1(const Sweep1Args a) {
    extern __shared__ __align__(128) unsigned char smraw1[];
    const SweepUnit u = a.units[blockIdx.x / NC];
    const unsigned rank = NC > 1 ? cluster_ctarank() : 0u, peer = rank ^ 1u;
    const int N = a.N, ld = a.ldD, nv = u.n, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int rpc = a.rows_per_chunk, n_chunks = (N + rpc - 1) / rpc;
    const int q0 = (NC > 1 && rank) ? (n_chunks + 1) / 2 : 0, q1 = (NC > 1 && !rank) ? (n_chunks + 1) / 2 : n_chunks, my_chunks = q1 - q0;
    const size_t chunk_bytes = (size_t)rpc * ld * 8;
    const int NS = a.ring_stages;
    unsigned char *ring = smraw1;
    cplx *X = reinterpret_cast<cplx *>(smraw1 + (size_t)NS * chunk_bytes);           // [2][NV][N]
    cplx *Ypart = X + (size_t)2 * NV * N;                                            // NC = 2: this CTA's partial sums [NV][N]
    __shared__ __align__(8) unsigned long long full[SW_STAGES], empty[SW_STAGES], xbar;
    __shared__ double red[SWEEP_NV][8];
    if (tid == 0) {
        for (int s = 0; s < SW_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], SW1_CONSUMERS / 32); }
        mbar_init(&xbar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (NC > 1) cluster_sync_all();                  // the peer's mbarrier exists before anything arrives on it
    if (warp == SW1_CONSUMERS / 32) {
        if (lane == 0) {
            const long long total = (long long)a.steps * 4 * my_chunks;
            for (long long g = 0; g < total; ++g) {
                const int slot = (int)(g % NS); const long long use = g / NS;
                if (use > 0) mbar_wait(&empty[slot], (unsigned)((use - 1) & 1));
                const int sst = (int)(g / my_chunks), q = q0 + (int)(g - (long long)sst * my_chunks), s = sst >> 2, st = sst & 3;
                const int li = 2 * s + (st == 0 ? 0 : (st == 3 ? 2 : 1));
                const int r0 = q * rpc, rows = min(rpc, N - r0);
                const double *src = a.D + ((size_t)u.group * a.n_idx + li) * (size_t)N * ld + (size_t)r0 * ld;
                const unsigned bytes = (unsigned)rows * ld * 8u;
                mbar_expect_tx(&full[slot], bytes);
                tma_bulk_g2s(ring + (size_t)slot * chunk_bytes, src, bytes, &full[slot]);
            }
        }
        if (NC > 1) cluster_sync_all();
        return;
    }
    // ---------------- consumers: thread tid owns rows tid + 224 t
    int row[NTILE], rowc[NTILE]; double eov[NTILE][NV];     // eps of the row's radial function / v of the trajectory
    cplx C[NTILE][NV], Acc[NTILE][NV], ph[NTILE][NV];
    double vinv[NV];
    #pragma unroll
    for (int q = 0; q < NV; ++q) vinv[q] = (q < nv) ? 1.0 / a.v[u.traj[q]] : 1.0;
    #pragma unroll
    for (int t = 0; t < NTILE; ++t) {
        row[t] = tid + SW1_CONSUMERS * t;
        const int rc = min(row[t], N - 1);
        rowc[t] = rc;
        const double e = a.eps[a.st_rad[rc]];
        #pragma unroll
        for (int q = 0; q < NV; ++q) {
            eov[t][q] = (q < nv) ? e / a.v[u.traj[q]] : 0.0;
            C[t][q] = cplx{0.0, 0.0}; Acc[t][q] = cplx{0.0, 0.0};
            if (q < nv && row[t] < N) { const double *src = a.C + ((size_t)u.traj[q] * N + row[t]) * 2; C[t][q] = cplx{src[0], src[1]}; }
        }
    }
    double drift[NV];
    #pragma unroll
    for (int q = 0; q < NV; ++q) drift[q] = (a.drift && q < nv) ? a.drift[u.traj[q]] : 0.0;
    const bool active = warp * 32 < N;                       // some lane of this warp owns a row
    auto phases = [&](double z) {
        #pragma unroll
        for (int t = 0; t < NTILE; ++t)
            #pragma unroll
            for (int q = 0; q < NV; ++q) { double sn, cs; sincos(eov[t][q] * z, &sn, &cs); ph[t][q] = cplx{cs, sn}; }
    };
    // x = P^H (C + alpha k) of this thread's rows into the stage-vector buffer `xb`
    auto put_x = [&](cplx *xb, double alpha, const cplx (&k)[NTILE][NV]) {
        #pragma unroll
        for (int t = 0; t < NTILE; ++t)
            if (row[t] < N) {
                #pragma unroll
                for (int q = 0; q < NV; ++q)
                    if (q < nv) xb[q * N + row[t]] = cmulc(cplx{C[t][q].x + alpha * k[t][q].x, C[t][q].y + alpha * k[t][q].y}, ph[t][q]);
            }
    };
    cplx kk[NTILE][NV];
    #pragma unroll
    for (int t = 0; t < NTILE; ++t)
        #pragma unroll
        for (int q = 0; q < NV; ++q) kk[t][q] = cplx{0.0, 0.0};
    phases(a.zh[0]);
    put_x(X, 0.0, kk);
    int xb = 0;
    long long g = 0;
    bar_sync(1, SW1_CONSUMERS);
    for (int s = 0; s < a.steps; ++s) {
        const double h = a.hs[s];
        #pragma unroll 1
        for (int st = 0; st < 4; ++st) {
            const cplx *Xc = X + (size_t)xb * NV * N;
            // ILP independent accumulator sets (consecutive streamed rows) when a thread has few (row, trajectory) pairs:
            // a single set would be one dependent fma chain of N links
            constexpr int ILP = (NTILE * NV <= 2) ? 4 : ((NTILE * NV <= 4) ? 2 : 1);
            cplx acc[ILP][NTILE][NV];
            #pragma unroll
            for (int i = 0; i < ILP; ++i)
                #pragma unroll
                for (int t = 0; t < NTILE; ++t)
                    #pragma unroll
                    for (int q = 0; q < NV; ++q) acc[i][t][q] = cplx{0.0, 0.0};
            for (int c = q0; c < q1; ++c) {
                const int slot = (int)(g % NS);
                mbar_wait(&full[slot], (unsigned)((g / NS) & 1));
                if (active) {
                    const double *buf = reinterpret_cast<const double *>(ring + (size_t)slot * chunk_bytes);
                    const int c0 = c * rpc, rows = min(rpc, N - c0);
                    auto one_row = [&](int rr, int set) {
                        const double *Dc = buf + (size_t)rr * ld;
                        cplx xq[NV];
                        #pragma unroll
                        for (int q = 0; q < NV; ++q) xq[q] = Xc[(q < nv ? q : 0) * N + c0 + rr];
                        #pragma unroll
                        for (int t = 0; t < NTILE; ++t) {
                            const double d = Dc[rowc[t]];
                            #pragma unroll
                            for (int q = 0; q < NV; ++q) { acc[set][t][q].x = fma(d, xq[q].x, acc[set][t][q].x); acc[set][t][q].y = fma(d, xq[q].y, acc[set][t][q].y); }
                        }
                    };
                    int rr = 0;
                    for (; rr + 4 <= rows; rr += 4) {
                        one_row(rr, 0); one_row(rr + 1, 1 % ILP); one_row(rr + 2, 2 % ILP); one_row(rr + 3, 3 % ILP);
                    }
                    for (; rr < rows; ++rr) one_row(rr, 0);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[slot]);
                ++g;
            }
            #pragma unroll
            for (int i = 1; i < ILP; ++i)
                #pragma unroll
                for (int t = 0; t < NTILE; ++t)
                    #pragma unroll
                    for (int q = 0; q < NV; ++q) { acc[0][t][q].x += acc[i][t][q].x; acc[0][t][q].y += acc[i][t][q].y; }
            if (NC > 1) {
                // add the peer CTA's partial sums (a + b = b + a: both CTAs carry bit-identical vectors)
                #pragma unroll
                for (int t = 0; t < NTILE; ++t)
                    if (row[t] < N) {
                        #pragma unroll
                        for (int q = 0; q < NV; ++q) Ypart[q * N + row[t]] = acc[0][t][q];
                    }
                bar_sync(1, SW1_CONSUMERS);                  // every partial sum of this CTA is written; every read of the previous stage is done
                if (tid == 0) mbar_arrive_peer(&xbar, peer);
                mbar_wait_cluster(&xbar, (unsigned)((s * 4 + st) & 1));
                #pragma unroll
                for (int t = 0; t < NTILE; ++t)
                    if (row[t] < N) {
                        #pragma unroll
                        for (int q = 0; q < NV; ++q) { const cplx o = ld_peer(Ypart + q * N + row[t], peer); acc[0][t][q].x += o.x; acc[0][t][q].y += o.y; }
                    }
            }
            // k = -(i/v) P y; RK4 accumulation; the next stage's vector goes into the other buffer
            const double wgt = (st == 0 || st == 3) ? 1.0 : 2.0;
            #pragma unroll
            for (int t = 0; t < NTILE; ++t)
                #pragma unroll
                for (int q = 0; q < NV; ++q) {
                    const cplx y = cmul(acc[0][t][q], ph[t][q]);
                    kk[t][q] = cplx{y.y * vinv[q], -y.x * vinv[q]};
                    Acc[t][q].x += wgt * kk[t][q].x; Acc[t][q].y += wgt * kk[t][q].y;
                    if (st == 3) { C[t][q].x += (h / 6.0) * Acc[t][q].x; C[t][q].y += (h / 6.0) * Acc[t][q].y; Acc[t][q] = cplx{0.0, 0.0}; }
                }
            // stage st + 1 (or stage 0 of the next step): position and alpha
            const bool last = (st == 3 && s + 1 == a.steps);
            if (!last) {
                const int nst = (st + 1) & 3, ns = s + (st == 3);
                const int li = 2 * ns + (nst == 0 ? 0 : (nst == 3 ? 2 : 1));
                if (st == 0 || st == 2) phases(a.zh[li]);            // the position changes at z -> z_mid and z_mid -> z_new
                const double hn = (st == 3) ? 0.0 : h;
                const double alpha = (nst == 0) ? 0.0 : (nst == 3 ? hn : 0.5 * hn);
                put_x(X + (size_t)(xb ^ 1) * NV * N, alpha, kk);
            }
            xb ^= 1;
            bar_sync(1, SW1_CONSUMERS);
        }
        if (a.drift) {
            #pragma unroll
            for (int q = 0; q < NV; ++q) {
                double part = 0.0;
                #pragma unroll
                for (int t = 0; t < NTILE; ++t) if (row[t] < N) part += C[t][q].x * C[t][q].x + C[t][q].y * C[t][q].y;
                part = warp_sum(part);
                if (lane == 0) red[q][warp] = part;
            }
            bar_sync(1, SW1_CONSUMERS);
            #pragma unroll
            for (int q = 0; q < NV; ++q) {
                double tot = 0.0;
                for (int w = 0; w < SW1_CONSUMERS / 32; ++w) tot += red[q][w];
                drift[q] = fmax(drift[q], fabs(tot - 1.0));
            }
            bar_sync(1, SW1_CONSUMERS);
        }
    }
    if (NC > 1) cluster_sync_all();                  // neither CTA leaves while the other may still read its partial sums
    if (rank != 0) return;
    #pragma unroll
    for (int q = 0; q < NV; ++q)
        if (q < nv) {
            #pragma unroll
            for (int t = 0; t < NTILE; ++t)
                if (row[t] < N) { double *dst = a.C + ((size_t)u.traj[q] * N + row[t]) * 2; dst[0] = C[t][q].x; dst[1] = C[t][q].y; }
            if (a.drift && tid == 0) a.drift[u.traj[q]] = drift[q];
        }
}

// ------------------------------------------------------------------ a7, large N_P: blocked Gauss-Jordan in global memory
// In-place inversion of the n x n matrix G (row-major, global / L2) in panels of FJ_NB columns.  A panel is
// eliminated in shared memory exactly as the unblocked algorithm does it (partial pivoting over the rows not yet
// used); its row interchanges are then applied to the other columns, and with W = the (interchanged) pivot rows
// the rest of the matrix is updated in ONE pass,  G[i][c] = (i in panel ? 0 : G[i][c]) + sum_t Pn[i][t] W[t][c],
// which is the block form of the same FJ_NB elimination steps (traffic over G: once per panel, not once per step).
constexpr int FJ_NB = 8;

__device__ void gauss_jordan_blocked(cplx *G, int n, cplx *Pn /*[n][FJ_NB]*/, cplx *W /*[FJ_NB][n]*/, cplx *col /*[n]*/,
                                     int *piv /*[n]*/, int *s_piv, int *s_flag) {
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5;
    __shared__ cplx rowv[FJ_NB];
    for (int j0 = 0; j0 < n; j0 += FJ_NB) {
        const int w = min(FJ_NB, n - j0);
        for (int e = tid; e < n * w; e += nt) { const int i = e / w, t = e - i * w; Pn[i * FJ_NB + t] = G[(size_t)i * n + j0 + t]; }
        __syncthreads();
        for (int t = 0; t < w; ++t) {
            const int j = j0 + t;
            if (warp == 0) {
                double best = -1.0; int bi = j;
                for (int i = j + lane; i < n; i += 32) { const cplx x = Pn[i * FJ_NB + t]; const double m = x.x * x.x + x.y * x.y; if (m > best) { best = m; bi = i; } }
                #pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const double m2 = __shfl_xor_sync(0xffffffffu, best, o); const int i2 = __shfl_xor_sync(0xffffffffu, bi, o);
                    if (m2 > best || (m2 == best && i2 < bi)) { best = m2; bi = i2; }
                }
                if (lane == 0) { *s_piv = bi; piv[j] = bi; if (!(best > 0.0)) *s_flag = 1; }
            }
            __syncthreads();
            const int pr = *s_piv;
            if (pr != j) {
                if (tid < w) { const cplx x = Pn[j * FJ_NB + tid]; Pn[j * FJ_NB + tid] = Pn[pr * FJ_NB + tid]; Pn[pr * FJ_NB + tid] = x; }
                __syncthreads();
            }
            const cplx d = Pn[j * FJ_NB + t];
            const double dn = d.x * d.x + d.y * d.y;
            const cplx dinv = (dn > 0.0) ? cplx{d.x / dn, -d.y / dn} : cplx{0.0, 0.0};
            for (int i = tid; i < n; i += nt) col[i] = Pn[i * FJ_NB + t];
            if (tid < w) rowv[tid] = (tid == t) ? dinv : cmul(Pn[j * FJ_NB + tid], dinv);
            __syncthreads();
            for (int e = tid; e < n * w; e += nt) {
                const int i = e / w, tt = e - i * w;
                cplx v = Pn[i * FJ_NB + tt];
                if (tt == t) v = {0.0, 0.0};
                Pn[i * FJ_NB + tt] = (i == j) ? rowv[tt] : csub(v, cmul(col[i], rowv[tt]));
            }
            __syncthreads();
        }
        // the panel's row interchanges on the other columns, in order
        for (int t = 0; t < w; ++t) {
            const int j = j0 + t, pr = piv[j];
            if (pr != j) {
                for (int c = tid; c < n; c += nt)
                    if (c < j0 || c >= j0 + w) { const cplx x = G[(size_t)j * n + c]; G[(size_t)j * n + c] = G[(size_t)pr * n + c]; G[(size_t)pr * n + c] = x; }
                __syncthreads();
            }
        }
        for (int e = tid; e < w * n; e += nt) { const int t = e / n, c = e - t * n; W[e] = G[(size_t)(j0 + t) * n + c]; }
        __syncthreads();
        {
            int i = tid / n, c = tid - i * n;
            const int di = nt / n, dc = nt - di * n;
            for (int e = tid; e < n * n; e += nt) {
                if (c >= j0 && c < j0 + w) G[e] = Pn[i * FJ_NB + (c - j0)];
                else {
                    const cplx *pn = Pn + i * FJ_NB;
                    cplx acc = (i >= j0 && i < j0 + w) ? cplx{0.0, 0.0} : G[e];
                    for (int t = 0; t < w; ++t) { const cplx x = pn[t], y = W[t * n + c]; acc.x += x.x * y.x - x.y * y.y; acc.y += x.x * y.y + x.y * y.x; }
                    G[e] = acc;
                }
                i += di; c += dc; if (c >= n) { c -= n; ++i; }
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------ a7: Schur complement + inverse
// grid = positions; block = 512.  A = I - K K^H (row-major, ld = NP) lives in shared memory when it fits, else in
// the output buffer (global).  K is staged through shared memory in column chunks of odd width cw (conflict-free).
// A^{-1} by in-place Gauss-Jordan elimination with partial (row) pivoting, first maximal |pivot| wins; the row
// interchanges are undone as column interchanges in reverse order at the end.
struct FactorArgs { const double *K; double *Ainv; int *flags; int NT, NP, use_smem, cw; size_t out_stride; };

__global__ void __launch_bounds__(512) k_factor(const FactorArgs a) {
    extern __shared__ __align__(16) double sm[];
    const int n = a.NP, NT = a.NT, cw = a.cw, tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const size_t p = blockIdx.x;
    const cplx *K = reinterpret_cast<const cplx *>(a.K) + p * (size_t)n * NT;
    cplx *G = reinterpret_cast<cplx *>(a.Ainv) + p * a.out_stride;
    cplx *smc = reinterpret_cast<cplx *>(sm);
    cplx *A = a.use_smem ? smc : G;
    cplx *Kc = smc + (a.use_smem ? (size_t)n * n : 0);     // [n][cw]
    cplx *col = Kc + (size_t)n * cw, *rowj = col + n;      // [n] each
    int *piv = reinterpret_cast<int *>(rowj + n), *idx = piv + n;
    __shared__ int s_flag, s_piv;
    if (tid == 0) s_flag = 0;
    __syncthreads();
    // A[r][s] = delta_rs - sum_i K[r][i] conj(K[s][i]), accumulated in the order i = 0..NT-1 (the elimination order)
    int bad = 0;
    for (int i0 = 0; i0 < NT; i0 += cw) {
        const int w = min(cw, NT - i0);
        for (int e = tid; e < n * w; e += nt) {
            const int r = e / w, ii = e - r * w;
            const cplx k = K[(size_t)r * NT + i0 + ii];
            Kc[r * cw + ii] = k;
            if (!(k.x * k.x + k.y * k.y < 1.0)) bad = 1;       // pivot-order precondition |K_ij| < 1
        }
        __syncthreads();
        for (int e = tid; e < n * n; e += nt) {
            const int r = e / n, s = e - r * n;
            cplx acc = (i0 == 0) ? cplx{(r == s) ? 1.0 : 0.0, 0.0} : A[e];
            const cplx *Kr = Kc + r * cw, *Ks = Kc + s * cw;
            for (int ii = 0; ii < w; ++ii) { const cplx x = Kr[ii], y = Ks[ii]; acc.x -= x.x * y.x + x.y * y.y; acc.y -= x.y * y.x - x.x * y.y; }
            A[e] = acc;
        }
        __syncthreads();
    }
    if (bad) s_flag = 2;
    if (!a.use_smem) {
        // large N_P: the shared memory that staged K now holds the panel, the pivot rows and the column vector
        cplx *Pn = smc, *Wr = Pn + (size_t)n * FJ_NB, *colv = Wr + (size_t)n * FJ_NB;
        int *pivg = reinterpret_cast<int *>(colv + n);
        gauss_jordan_blocked(G, n, Pn, Wr, colv, pivg, &s_piv, &s_flag);
        for (int j = n - 1; j >= 0; --j) {
            const int q = pivg[j];
            if (q != j) {
                for (int r = tid; r < n; r += nt) { const cplx t = G[(size_t)r * n + j]; G[(size_t)r * n + j] = G[(size_t)r * n + q]; G[(size_t)r * n + q] = t; }
                __syncthreads();
            }
        }
        if (tid == 0 && s_flag) a.flags[p] = s_flag;
        return;
    }
    {   // shared-memory A: the same blocked elimination, panel buffers in the area that staged K (piv, idx lie behind it)
        cplx *Pn = Kc, *Wr = Pn + (size_t)n * FJ_NB, *colv = Wr + (size_t)n * FJ_NB;
        gauss_jordan_blocked(A, n, Pn, Wr, colv, piv, &s_piv, &s_flag);
    }
    if (a.use_smem) {
        if (tid == 0) {
            for (int c = 0; c < n; ++c) idx[c] = c;
            for (int j = n - 1; j >= 0; --j) { const int q = piv[j]; const int t = idx[j]; idx[j] = idx[q]; idx[q] = t; }
        }
        __syncthreads();
        for (int e = tid; e < n * n; e += nt) { const int r = e / n, c = e - r * n; G[e] = A[(size_t)r * n + idx[c]]; }
    } else {
        for (int j = n - 1; j >= 0; --j) {
            const int q = piv[j];
            if (q != j) {
                for (int r = tid; r < n; r += nt) { const cplx t = A[(size_t)r * n + j]; A[(size_t)r * n + j] = A[(size_t)r * n + q]; A[(size_t)r * n + q] = t; }
                __syncthreads();
            }
        }
    }
    if (tid == 0 && s_flag) a.flags[p] = s_flag;
}

// ------------------------------------------------------------------ a7, N_P <= 90: A and the elimination in registers
// grid = positions; block = 15 worker warps + 1 panel warp.  Worker (ty = warp, tx = lane) owns the elements
// A[ty + 15 r][tx + 32 s], r < 6, s < 3, in registers for the whole kernel: the Schur complement is accumulated there
// (K staged in shared memory, row stride odd), and the blocked Gauss-Jordan elimination (panels of FR_NB columns)
// updates them in place.  Rows are never interchanged: the pivot of column j is the largest entry among the rows not
// yet used (the same candidates, by row identity, as partial pivoting with interchanges; first maximal row wins), and
// with piv[j] = that row the inverse is  Ainv[pinv[r]][piv[k]] = G[r][k],  pinv[piv[j]] = j.
// The panel warp (lane owns rows lane, lane + 32, lane + 64) eliminates the FR_NB columns of a panel in registers
// with shuffles only; it works one panel ahead: the workers update and hand over the columns of panel p + 1 first,
// then finish the update of panel p while the panel warp eliminates panel p + 1.
constexpr int FR_WW = 15, FR_RN = 6, FR_CN = 3, FR_NMAX = FR_WW * FR_RN, FR_WORKERS = 32 * FR_WW, FR_THREADS = FR_WORKERS + 32;
constexpr int FR_NB = 4;                                              // panel width (the panel warp holds 3 rows of it per lane)
constexpr int FR_BAR_DONE = 1, FR_BAR_WORK = 2, FR_BAR_PANEL = 3;      // named barriers (0 is unused here)


// Gauss-Jordan steps j0 .. j0 + w - 1 on the panel Pn [n][FR_NB] (shared), by one warp, in registers.  The warp is
// alone on the critical path of the whole kernel, so a step is kept short: branch-free pivot search on integer
// keys (bit pattern of |x|^2 + 1 for a free row, 0 for a used one: the order of non-negative doubles) with three
// warp reductions, the pivot row passed through shared memory, one reciprocal, one update formula for every row
// and a fix-up of the pivot row by its owner.  usedmask: bit q = row lane + 32 q already used as a pivot.
__device__ __forceinline__ void fr_panel(cplx *Pn, const int n, const int w, const int j0, const int pid, unsigned &usedmask,
                                         int *piv, int *rowpid, int *rowslot, int *s_flag, cplx *rowbuf /*[2][FR_NB]*/, const int lane) {
    cplx p[3][FR_NB];
    #pragma unroll
    for (int q = 0; q < 3; ++q) {
        const int row = min(lane + 32 * q, n - 1);                    // rows >= n: copies, marked used by the caller
        #pragma unroll
        for (int t = 0; t < FR_NB; ++t) p[q][t] = Pn[row * FR_NB + t];
    }
    #pragma unroll
    for (int t = 0; t < FR_NB; ++t) {
        if (t < w) {
            unsigned long long best = 0; int brow = lane;
            #pragma unroll
            for (int q = 0; q < 3; ++q) {
                const double m = p[q][t].x * p[q][t].x + p[q][t].y * p[q][t].y;
                const unsigned long long key = ((usedmask >> q) & 1u) ? 0ull : (unsigned long long)__double_as_longlong(m) + 1ull;
                const bool gt = key > best;                           // first maximal row wins within the lane
                best = gt ? key : best; brow = gt ? lane + 32 * q : brow;
            }
            const unsigned hi = (unsigned)(best >> 32), lo = (unsigned)best;
            const unsigned H = __reduce_max_sync(0xffffffffu, hi);
            const unsigned L = __reduce_max_sync(0xffffffffu, hi == H ? lo : 0u);
            const int pr = (int)__reduce_min_sync(0xffffffffu, (hi == H && lo == L) ? (unsigned)brow : 0x7fffffffu);
            cplx *rb = rowbuf + (t & 1) * FR_NB;
            #pragma unroll
            for (int q = 0; q < 3; ++q)
                if (pr == lane + 32 * q) {                            // owner of the pivot row: predicated stores, no selects
                    #pragma unroll
                    for (int tt = 0; tt < FR_NB; ++tt) rb[tt] = p[q][tt];
                }
            __syncwarp();
            cplx rowv[FR_NB];
            #pragma unroll
            for (int tt = 0; tt < FR_NB; ++tt) rowv[tt] = rb[tt];
            const cplx d = rowv[t];
            const double dn = d.x * d.x + d.y * d.y;
            const double inv = (dn > 0.0) ? __drcp_rn(dn) : 0.0;
            const cplx dinv = {d.x * inv, -d.y * inv};
            #pragma unroll
            for (int tt = 0; tt < FR_NB; ++tt) rowv[tt] = (tt == t) ? dinv : cmul(rowv[tt], dinv);
            #pragma unroll
            for (int q = 0; q < 3; ++q) {
                const cplx col = p[q][t];
                #pragma unroll
                for (int tt = 0; tt < FR_NB; ++tt) {                  // v - col * rowv as two fma chains
                    const cplx v = (tt == t) ? cplx{0.0, 0.0} : p[q][tt];
                    p[q][tt].x = fma(col.y, rowv[tt].y, fma(-col.x, rowv[tt].x, v.x));
                    p[q][tt].y = fma(-col.y, rowv[tt].x, fma(-col.x, rowv[tt].y, v.y));
                }
            }
            #pragma unroll
            for (int q = 0; q < 3; ++q)
                if (pr == lane + 32 * q) {                            // the pivot row itself
                    #pragma unroll
                    for (int tt = 0; tt < FR_NB; ++tt) p[q][tt] = rowv[tt];
                    usedmask |= 1u << q;
                }
            if (lane == 0) {
                piv[j0 + t] = pr; rowpid[pr] = pid; rowslot[pr] = t;
                const double mbest = __longlong_as_double((long long)((((unsigned long long)H << 32) | L) - 1ull));
                if (!(mbest > 0.0) || H >= 0x7ff00000u) *s_flag = 1;   // zero, infinite or NaN pivot
            }
        }
    }
    #pragma unroll
    for (int q = 0; q < 3; ++q) {
        const int row = lane + 32 * q;
        if (row < n) {
            #pragma unroll
            for (int t = 0; t < FR_NB; ++t) Pn[row * FR_NB + t] = (t < w) ? p[q][t] : cplx{0.0, 0.0};
        }
    }
}

__global__ void __launch_bounds__(FR_THREADS, 1) k_factor_reg(const FactorArgs a) {
    extern __shared__ __align__(16) double sm[];
    const int n = a.NP, NT = a.NT, cw = a.cw, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t pos = blockIdx.x;
    cplx *Ks = reinterpret_cast<cplx *>(sm);                          // [n][cw] K chunk
    cplx *Pn = Ks + (size_t)n * cw;                                  // [2][FR_NMAX][FR_NB]
    cplx *W = Pn + 2 * FR_NMAX * FR_NB;                               // [FR_NB][FR_NMAX]
    int *piv = reinterpret_cast<int *>(W + FR_NB * FR_NMAX), *pinv = piv + FR_NMAX, *rowpid = pinv + FR_NMAX, *rowslot = rowpid + FR_NMAX;
    __shared__ int s_flag;
    __shared__ cplx rowbuf[2 * FR_NB];
    const int np = (n + FR_NB - 1) / FR_NB;

    if (warp == FR_WORKERS / 32) {                                    // ---- panel warp
        unsigned usedmask = 0;
        #pragma unroll
        for (int q = 0; q < 3; ++q) if (lane + 32 * q >= n) usedmask |= 1u << q;
        for (int p = 0; p < np; ++p) {
            bar_sync(FR_BAR_PANEL, FR_THREADS);
            fr_panel(Pn + (p & 1) * FR_NMAX * FR_NB, n, min(FR_NB, n - p * FR_NB), p * FR_NB, p, usedmask, piv, rowpid, rowslot, &s_flag, rowbuf, lane);
            bar_sync(FR_BAR_DONE, FR_THREADS);
        }
        return;
    }
    // ---- workers
    const int ty = warp, tx = lane;
    const cplx *K = reinterpret_cast<const cplx *>(a.K) + pos * (size_t)n * NT;
    cplx *G = reinterpret_cast<cplx *>(a.Ainv) + pos * a.out_stride;
    int rc[FR_RN], cc[FR_CN];                                         // clamped: out-of-range copies are computed, never stored
    #pragma unroll
    for (int r = 0; r < FR_RN; ++r) rc[r] = min(ty + FR_WW * r, n - 1);
    #pragma unroll
    for (int s = 0; s < FR_CN; ++s) cc[s] = min(tx + 32 * s, n - 1);
    if (tid == 0) s_flag = 0;
    if (tid < FR_NMAX) rowpid[tid] = -1;
    cplx acc[FR_RN][FR_CN];
    #pragma unroll
    for (int r = 0; r < FR_RN; ++r)
        #pragma unroll
        for (int s = 0; s < FR_CN; ++s) acc[r][s] = cplx{(rc[r] == cc[s]) ? 1.0 : 0.0, 0.0};
    // A[r][s] = delta_rs - sum_i K[r][i] conj(K[s][i]), i ascending (the elimination order)
    int bad = 0;
    for (int i0 = 0; i0 < NT; i0 += cw) {
        const int w = min(cw, NT - i0);
        if (i0) bar_sync(FR_BAR_WORK, FR_WORKERS);
        for (int e = tid; e < n * w; e += FR_WORKERS) {
            const int r = e / w, ii = e - r * w;
            const cplx k = K[(size_t)r * NT + i0 + ii];
            Ks[r * cw + ii] = k;
            if (!(k.x * k.x + k.y * k.y < 1.0)) bad = 1;              // pivot-order precondition |K_ij| < 1
        }
        bar_sync(FR_BAR_WORK, FR_WORKERS);
        #pragma unroll 1
        for (int ii = 0; ii < w; ++ii) {
            cplx kr[FR_RN], ks[FR_CN];
            #pragma unroll
            for (int r = 0; r < FR_RN; ++r) kr[r] = Ks[rc[r] * cw + ii];
            #pragma unroll
            for (int s = 0; s < FR_CN; ++s) ks[s] = Ks[cc[s] * cw + ii];
            #pragma unroll
            for (int r = 0; r < FR_RN; ++r)
                #pragma unroll
                for (int s = 0; s < FR_CN; ++s) {
                    acc[r][s].x = fma(-kr[r].y, ks[s].y, fma(-kr[r].x, ks[s].x, acc[r][s].x));     // two fma per component
                    acc[r][s].y = fma(kr[r].x, ks[s].y, fma(-kr[r].y, ks[s].x, acc[r][s].y));
                }
        }
    }
    if (bad) s_flag = 2;

    // hand the columns of panel q to the panel warp
    auto write_panel = [&](const int q) {
        const int j0 = q * FR_NB, wq = min(FR_NB, n - j0);
        cplx *P = Pn + (q & 1) * FR_NMAX * FR_NB;
        #pragma unroll
        for (int s = 0; s < FR_CN; ++s) {
            const int t = tx + 32 * s - j0;
            if (t >= 0 && t < wq) {
                #pragma unroll
                for (int r = 0; r < FR_RN; ++r) if (ty + FR_WW * r < n) P[(ty + FR_WW * r) * FR_NB + t] = acc[r][s];
            }
        }
        bar_arrive(FR_BAR_PANEL, FR_THREADS);                         // orders the stores above for the waiting panel warp
    };
    write_panel(0);
    bool pivrow[FR_RN];
    for (int p = 0; p < np; ++p) {
        const int j0 = p * FR_NB, w = min(FR_NB, n - j0);
        const cplx *P = Pn + (p & 1) * FR_NMAX * FR_NB;
        bar_sync(FR_BAR_DONE, FR_THREADS);                            // panel p eliminated: P, piv, rowpid
        #pragma unroll
        for (int r = 0; r < FR_RN; ++r) {                             // W[t][:] = row piv[j0 + t] before the update
            const int row = ty + FR_WW * r;
            pivrow[r] = row < n && rowpid[rc[r]] == p;
            if (pivrow[r]) {
                const int t = rowslot[row];
                #pragma unroll
                for (int s = 0; s < FR_CN; ++s) if (tx + 32 * s < n) W[t * FR_NMAX + tx + 32 * s] = acc[r][s];
            }
        }
        bar_sync(FR_BAR_WORK, FR_WORKERS);
        #pragma unroll
        for (int r = 0; r < FR_RN; ++r)
            if (pivrow[r]) {                                          // pivot rows of this panel start from zero
                #pragma unroll
                for (int s = 0; s < FR_CN; ++s) acc[r][s] = cplx{0.0, 0.0};
            }
        auto update_col = [&](const int s) {
            for (int t = 0; t < w; ++t) {
                const cplx y = W[t * FR_NMAX + cc[s]];
                #pragma unroll
                for (int r = 0; r < FR_RN; ++r) {
                    const cplx x = P[rc[r] * FR_NB + t];
                    acc[r][s].x = fma(-x.y, y.y, fma(x.x, y.x, acc[r][s].x)); acc[r][s].y = fma(x.y, y.x, fma(x.x, y.y, acc[r][s].y));
                }
            }
            const int t = tx + 32 * s - j0;
            if (t >= 0 && t < w) {                                    // the panel's own columns
                #pragma unroll
                for (int r = 0; r < FR_RN; ++r) acc[r][s] = P[rc[r] * FR_NB + t];
            }
        };
        // the column slab that holds the next panel goes first (three copies: register indices stay static)
        const int sn = (p + 1 < np) ? (j0 + FR_NB) >> 5 : -1;
        if (sn == 1)      { update_col(1); write_panel(p + 1); update_col(0); update_col(2); }
        else if (sn == 2) { update_col(2); write_panel(p + 1); update_col(0); update_col(1); }
        else              { update_col(0); if (sn == 0) write_panel(p + 1); update_col(1); update_col(2); }
    }
    // Ainv[pinv[r]][piv[k]] = G[r][k]: a lane's columns piv[tx + 32 s] are consecutive wherever the pivots stayed on
    // the diagonal, so the stores are mostly whole 512-byte runs; they drain while the next CTA starts
    if (tid < n) pinv[piv[tid]] = tid;
    bar_sync(FR_BAR_WORK, FR_WORKERS);
    #pragma unroll
    for (int r = 0; r < FR_RN; ++r)
        #pragma unroll
        for (int s = 0; s < FR_CN; ++s)
            if (ty + FR_WW * r < n && tx + 32 * s < n) G[(size_t)pinv[ty + FR_WW * r] * n + piv[tx + 32 * s]] = acc[r][s];
    if (tid == 0 && s_flag) a.flags[pos] = s_flag;
}

// ------------------------------------------------------------------ two-centre sweep
// grid = trajectories; block = 8 consumer warps + 1 producer warp.  Per RK4 stage, with the phase-free H0, K of the
// stage's position and the factorised Schur complement A = I - K K^H (a7):
//     y = H0 x;   y_P -= K y_T;   w_P = A^{-1} y_P;   w_T = y_T - K^H w_P;   k = -(i/v) P w.
// A^{-1} y_P: SOLVE = false: explicit inverse, one matrix-vector product;  SOLVE = true: blocked Cholesky factor
// (CholLayout, sweep.cuh), forward solve over the block rows of Lr, backward solve over the block columns of Lc.
// The matrices do not depend on the amplitudes, so the producer warp streams them through a shared-memory ring with TMA
// bulk copies (one per chunk), running ahead of the consumers across stage boundaries.  Chunk order of one RK4 step:
// stages 0..3 each [H rows | K rows | factor | K rows], then (drift only) K rows; producer and consumers walk the same
// loops (SweepSched gives the chunk shapes).
struct SweepSched {
    int N, NT, NP, rH, rK, rA, nH, nK, nA, nKT, cb;       // rA also: rows of K^T [NT][NP] per chunk (nKT chunks)
    __device__ SweepSched(int NT_, int NP_, int chunk_bytes) {
        NT = NT_; NP = NP_; N = NT + NP; cb = chunk_bytes;
        rH = max(1, chunk_bytes / (16 * N)); rK = max(1, chunk_bytes / (16 * NT)); rA = max(1, chunk_bytes / (16 * NP));
        nH = (N + rH - 1) / rH; nK = (NP + rK - 1) / rK; nA = (NP + rA - 1) / rA; nKT = (NT + rA - 1) / rA;
    }
    __device__ int rows_fwd(const CholLayout &L, int j) const { return max(1, min(L.nb(j), cb / (16 * L.len(j)))); }   // rows of block row j per chunk
    __device__ int rows_bwd(const CholLayout &L, int j) const { return max(1, cb / (16 * L.nb(j))); }                  // rows below block j per chunk
};

// sum over c of row[c] * x[c], c = 0..n-1, by one warp (every lane returns the sum)
__device__ __forceinline__ cplx warp_dot(const cplx *row, const cplx *x, int n, int lane) {
    double sr = 0.0, si = 0.0;
    for (int c = lane; c < n; c += 32) { const cplx k = row[c], v = x[c]; sr += k.x * v.x - k.y * v.y; si += k.x * v.y + k.y * v.x; }
    return {warp_sum(sr), warp_sum(si)};
}

constexpr int SW_DLD = CHOL_NB + 1;      // row stride of the staged diagonal block

constexpr int SW_TCOLS = 4;            // columns / rows of K per consumer thread in the K^H and K products: N_T, N_P <= 1024
constexpr int SW_TROWS = 8;            // rows of H0 per consumer thread: N <= 2048

// NC = 2: a cluster of two CTAs per trajectory.  Both hold the whole state and walk the same stages; the three matrix-vector
// products of a stage (H0 x, K y_T, K^H w_P) are split by streamed rows -- each CTA streams and multiplies one half of H0^T, K^T
// and K, i.e. half of the bytes that bound a single SM (its TMA stream and its shared-memory port) -- and the partial sums are
// exchanged through distributed shared memory (one mbarrier hand-shake per product; a + b = b + a, so both CTAs carry bit-identical
// vectors).  The triangular solves are done by both (no exchange inside the block recurrences).
template <bool SOLVE, int TR, int NC>  // TR = ceil(N / 256): rows of H0 per consumer thread
__global__ void __launch_bounds__(SW_CONSUMERS + 32, 1) k_sweep2(const Sweep2Args a, const int chunk_bytes, const int NS) {
    extern __shared__ __align__(128) unsigned char smraw[];
    const int NT = a.NT, NP = a.NP, N = NT + NP, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int t = blockIdx.x / NC;
    const unsigned rank = NC > 1 ? cluster_ctarank() : 0u;
    const bool track = a.drift != nullptr;
    const SweepSched S(NT, NP, chunk_bytes);
    const CholLayout CL(NP);
    unsigned char *ring = smraw;
    // shared: the stage vectors X, Y, w_P; the state of element j = tid + 256 t (amplitude C, RK4 accumulator, last slope,
    // phase) lives in registers of the thread that owns it
    cplx *X = reinterpret_cast<cplx *>(smraw + (size_t)NS * chunk_bytes);
    cplx *Y = X + N, *Wp = Y + N;
    cplx *Tj = Wp + NP, *Dblk = Tj + CHOL_NB, *part2 = Dblk + CHOL_NB * SW_DLD;                                  // SOLVE: [32], [32][33], [8][32]
    cplx *Ypart = part2 + 8 * CHOL_NB, *Kpart = Ypart + N, *Tpart = Kpart + NP;                                  // NC = 2: this CTA's partial sums [N], [NP], [NT]
    __shared__ __align__(8) unsigned long long full[SW_STAGES], empty[SW_STAGES], xbar[3];
    __shared__ double red[8];
    __shared__ int redi[8];
    if (tid == 0) {
        for (int s = 0; s < SW_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], SW_CONSUMERS / 32); }
        for (int s = 0; s < 3; ++s) mbar_init(&xbar[s], NC > 1 ? NC - 1 : 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (NC > 1) cluster_sync_all();                  // the peer's mbarriers exist before anything arrives on them
    // chunk ranges of this CTA in the three split products
    const int hH = (S.nH + NC - 1) / NC, hKT = (S.nKT + NC - 1) / NC, hK = (S.nK + NC - 1) / NC;
    const int qH0 = min(S.nH, (int)rank * hH), qH1 = min(S.nH, qH0 + hH);
    const int qT0 = min(S.nKT, (int)rank * hKT), qT1 = min(S.nKT, qT0 + hKT);
    const int qK0 = min(S.nK, (int)rank * hK), qK1 = min(S.nK, qK0 + hK);
    const cplx *Hg = reinterpret_cast<const cplx *>(a.H), *Kg = reinterpret_cast<const cplx *>(a.K), *Ag = reinterpret_cast<const cplx *>(a.Ainv);
    const cplx *KTg = reinterpret_cast<const cplx *>(a.KT);
    const size_t a_stride = wp_factor_elems(NP);

    if (warp == SW_CONSUMERS / 32) {
        // ---------------- producer: one lane streams the chunk sequence of the whole window
        if (lane != 0) { if (NC > 1) cluster_sync_all(); return; }
        long long g = 0;
        auto push = [&](const cplx *src, unsigned bytes) {
            const int slot = (int)(g % NS); const long long use = g / NS;
            if (use > 0) mbar_wait(&empty[slot], (unsigned)((use - 1) & 1));
            mbar_expect_tx(&full[slot], bytes);
            tma_bulk_g2s(ring + (size_t)slot * chunk_bytes, src, bytes, &full[slot]);
            ++g;
        };
        auto push_K = [&](const cplx *Kp) { for (int q = qK0; q < qK1; ++q) { const int r0 = q * S.rK, rows = min(S.rK, NP - r0); push(Kp + (size_t)r0 * NT, (unsigned)rows * NT * 16u); } };
        auto push_KT = [&](const cplx *Kp, int q0, int q1) { for (int q = q0; q < q1; ++q) { const int r0 = q * S.rA, rows = min(S.rA, NT - r0); push(Kp + (size_t)r0 * NP, (unsigned)rows * NP * 16u); } };
        for (int s = 0; s < a.steps; ++s)
            for (int st = 0; st < (track ? 5 : 4); ++st) {
                const int li = 2 * s + (st == 0 ? 0 : (st >= 3 ? 2 : 1));
                const size_t pos = (size_t)t * a.n_idx + li;
                const cplx *Kp = Kg + pos * (size_t)NP * NT, *KTp = KTg + pos * (size_t)NP * NT;
                if (st == 4) { push_KT(KTp, 0, S.nKT); break; }             // the norm is formed by both CTAs in full
                const cplx *Hp = Hg + pos * (size_t)N * N, *Ap = Ag + pos * a_stride;
                for (int q = qH0; q < qH1; ++q) { const int r0 = q * S.rH, rows = min(S.rH, N - r0); push(Hp + (size_t)r0 * N, (unsigned)rows * N * 16u); }
                push_KT(KTp, qT0, qT1);
                if (!SOLVE) {
                    for (int q = 0; q < S.nA; ++q) { const int r0 = q * S.rA, rows = min(S.rA, NP - r0); push(Ap + (size_t)r0 * NP, (unsigned)rows * NP * 16u); }
                } else {
                    for (int j = 0; j < CL.nblk; ++j) {                                   // forward: block rows of Lr
                        const int nbj = CL.nb(j), len = CL.len(j), rf = S.rows_fwd(CL, j);
                        for (int r0 = 0; r0 < nbj; r0 += rf) push(Ap + CL.off_r(j) + (size_t)r0 * len, (unsigned)min(rf, nbj - r0) * len * 16u);
                    }
                    for (int j = CL.nblk - 1; j >= 0; --j) {                              // backward: block columns of Lc, the part below first
                        const int nbj = CL.nb(j), below = NP - CHOL_NB * j - nbj, rb = S.rows_bwd(CL, j);
                        for (int r0 = 0; r0 < below; r0 += rb) push(Ap + CL.off_c(j) + (size_t)(nbj + r0) * nbj, (unsigned)min(rb, below - r0) * nbj * 16u);
                        push(Ap + CL.off_c(j), (unsigned)nbj * nbj * 16u);
                    }
                }
                push_K(Kp);
            }
        if (NC > 1) cluster_sync_all();
        return;
    }
    // ---------------- consumers (256 threads)
    const double vel = a.v[t];
    cplx C[TR], Acc[TR], Kn[TR], ph[TR]; double eov[TR];
    #pragma unroll
    for (int tr = 0; tr < TR; ++tr) {
        const int j = tid + SW_CONSUMERS * tr;
        C[tr] = Acc[tr] = Kn[tr] = ph[tr] = cplx{0.0, 0.0}; eov[tr] = 0.0;
        if (j < N) {
            const double *src = a.C + ((size_t)t * N + j) * 2;
            C[tr] = cplx{src[0], src[1]};
            eov[tr] = ((j < NT) ? a.eps_T[a.st_rad_T[j]] : a.eps_P[a.st_rad_P[j - NT]]) / vel;
        }
    }
    int li_ph = -1;                                          // half-step index the phases in ph[] belong to
    // first position of this window whose overlap factorisation failed (n_idx: none)
    int first_bad = a.n_idx;
    if (a.flags) {
        for (int li = tid; li < a.n_idx; li += SW_CONSUMERS) if (a.flags[(size_t)t * a.n_idx + li]) first_bad = min(first_bad, li);
        first_bad = __reduce_min_sync(0xffffffffu, first_bad);
        if (lane == 0) redi[warp] = first_bad;
    }
    double drift = track ? a.drift[t] : 0.0;
    long long g = 0;                                         // chunk counter, in step with the producer
    auto acquire = [&]() -> const cplx * {
        const int slot = (int)(g % NS);
        mbar_wait(&full[slot], (unsigned)((g / NS) & 1));
        return reinterpret_cast<const cplx *>(ring + (size_t)slot * chunk_bytes);
    };
    auto release = [&]() {
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[(int)(g % NS)]);
        ++g;
    };
    consumer_sync();
    if (a.flags) { for (int w = 0; w < 8; ++w) first_bad = min(first_bad, redi[w]); }
    // NC = 2: add the peer CTA's partial sums to this thread's (elements tid + 256 k < n); `buf` is this CTA's copy of them
    unsigned xphase = 0;                                     // bit w: parity of the next wait on xbar[w]
    auto exchange = [&](cplx *val, int nval, int n, cplx *buf, int which) {
        for (int k = 0; k < nval; ++k) { const int j = tid + SW_CONSUMERS * k; if (j < n) buf[j] = val[k]; }
        consumer_sync();                                     // every partial sum of this CTA is in `buf` (and every read of the previous exchange is done)
        if (tid < NC && tid != (int)rank) mbar_arrive_peer(&xbar[which], (unsigned)tid);
        mbar_wait_cluster(&xbar[which], (xphase >> which) & 1u);
        xphase ^= 1u << which;
        // summed in rank order by every CTA of the cluster: bit-identical vectors everywhere
        for (int k = 0; k < nval; ++k) {
            const int j = tid + SW_CONSUMERS * k;
            if (j < n) {
                cplx sum = {0.0, 0.0};
                #pragma unroll
                for (int r = 0; r < NC; ++r) { const cplx o = (r == (int)rank) ? buf[j] : ld_peer(buf + j, (unsigned)r); sum.x += o.x; sum.y += o.y; }
                val[k] = sum;
            }
        }
    };

    for (int s = 0; s < a.steps; ++s) {
        const double h = a.hs[s];
        #pragma unroll 1
        for (int st = 0; st < 5; ++st) {
            // st = 0..3: RK4 stages; st = 4: norm c^H S c at z_new (only when drift is tracked)
            if (st == 4 && !track) break;
            const int li = 2 * s + (st == 0 ? 0 : (st >= 3 ? 2 : 1));
            const double alpha = (st == 0 || st == 4) ? 0.0 : (st == 3 ? h : 0.5 * h);
            const double wgt = (st == 0 || st == 3) ? 1.0 : 2.0;
            const double z = a.zh[li];
            #pragma unroll
            for (int tr = 0; tr < TR; ++tr) {
                const int j = tid + SW_CONSUMERS * tr;
                if (li != li_ph) { double sn, cs; sincos(eov[tr] * z, &sn, &cs); ph[tr] = cplx{cs, sn}; }
                if (j < N) X[j] = cmulc(cplx{C[tr].x + alpha * Kn[tr].x, C[tr].y + alpha * Kn[tr].y}, ph[tr]);
            }
            li_ph = li;
            consumer_sync();
            // (K v)_r = sum_c K^T[c][r] v_c for this thread's rows r = tid + 256 t of the projectile block: the rows c of K^T stream
            // through the ring, v_c is a broadcast, consecutive lanes read consecutive elements -- no reduction
            // (ILP independent accumulator sets over consecutive streamed rows: one set is a dependent fma chain of N_T links)
            auto k_times = [&](const cplx *vT, cplx (&accK)[SW_TCOLS], int q0, int q1) {
                constexpr int TC = (TR + 1) / 2, ILP = TC == 1 ? 4 : 2;
                cplx ak[ILP][TC];
                #pragma unroll
                for (int u = 0; u < ILP; ++u)
                    #pragma unroll
                    for (int tc = 0; tc < TC; ++tc) ak[u][tc] = cplx{0.0, 0.0};
                for (int q = q0; q < q1; ++q) {
                    const cplx *buf = acquire();
                    const int c0 = q * S.rA, rows = min(S.rA, NT - c0);
                    auto one = [&](int rr, int u) {
                        const cplx y = vT[c0 + rr];
                        const cplx *Kc = buf + (size_t)rr * NP;
                        #pragma unroll
                        for (int tc = 0; tc < TC; ++tc) {
                            const int r = tid + SW_CONSUMERS * tc;
                            if (r < NP) { const cplx k = Kc[r]; ak[u][tc].x += k.x * y.x - k.y * y.y; ak[u][tc].y += k.x * y.y + k.y * y.x; }
                        }
                    };
                    int rr = 0;
                    for (; rr + ILP <= rows; rr += ILP) {
                        #pragma unroll
                        for (int u = 0; u < ILP; ++u) one(rr + u, u);
                    }
                    for (; rr < rows; ++rr) one(rr, 0);
                    release();
                }
                #pragma unroll
                for (int tc = 0; tc < SW_TCOLS; ++tc) {
                    accK[tc] = cplx{0.0, 0.0};
                    if (tc < TC) {
                        #pragma unroll
                        for (int u = 0; u < ILP; ++u) { accK[tc].x += ak[u][tc < TC ? tc : 0].x; accK[tc].y += ak[u][tc < TC ? tc : 0].y; }
                    }
                }
            };
            if (st == 4) {
                // c^H S c = |c|^2 + 2 Re( X_P^H K X_T )
                cplx accK[SW_TCOLS];
                k_times(X, accK, 0, S.nKT);
                double nrm = 0.0;
                #pragma unroll
                for (int tc = 0; tc < SW_TCOLS; ++tc) {
                    const int r = tid + SW_CONSUMERS * tc;
                    if (r < NP) nrm += 2.0 * (X[NT + r].x * accK[tc].x + X[NT + r].y * accK[tc].y);
                }
                #pragma unroll
                for (int tr = 0; tr < TR; ++tr) { const int j = tid + SW_CONSUMERS * tr; if (j < N) nrm += X[j].x * X[j].x + X[j].y * X[j].y; }
                nrm = warp_sum(nrm);
                if (lane == 0) red[warp] = nrm;
                consumer_sync();
                double tot = 0.0;
                for (int w = 0; w < 8; ++w) tot += red[w];
                drift = fmax(drift, fabs(tot - 1.0));
                consumer_sync();
                break;
            }
            // y = H0 x from the streamed rows c of H0^T: y_r = sum_c H0^T[c][r] x_c, thread tid owns the rows r = tid + 256 t
            {
                constexpr int ILP = TR == 1 ? 4 : (TR <= 3 ? 2 : 1);
                cplx accY[ILP][TR];
                #pragma unroll
                for (int u = 0; u < ILP; ++u)
                    #pragma unroll
                    for (int tr = 0; tr < TR; ++tr) accY[u][tr] = cplx{0.0, 0.0};
                for (int q = qH0; q < qH1; ++q) {
                    const cplx *buf = acquire();
                    const int c0 = q * S.rH, rows = min(S.rH, N - c0);
                    auto one = [&](int rr, int u) {
                        const cplx x = X[c0 + rr];
                        const cplx *Hc = buf + (size_t)rr * N;
                        #pragma unroll
                        for (int tr = 0; tr < TR; ++tr) {
                            const int r = tid + SW_CONSUMERS * tr;
                            if (r < N) { const cplx hh = Hc[r]; accY[u][tr].x += hh.x * x.x - hh.y * x.y; accY[u][tr].y += hh.x * x.y + hh.y * x.x; }
                        }
                    };
                    int rr = 0;
                    for (; rr + ILP <= rows; rr += ILP) {
                        #pragma unroll
                        for (int u = 0; u < ILP; ++u) one(rr + u, u);
                    }
                    for (; rr < rows; ++rr) one(rr, 0);
                    release();
                }
                #pragma unroll
                for (int tr = 0; tr < TR; ++tr) {
                    #pragma unroll
                    for (int u = 1; u < ILP; ++u) { accY[0][tr].x += accY[u][tr].x; accY[0][tr].y += accY[u][tr].y; }
                }
                if (NC > 1) exchange(accY[0], TR, N, Ypart, 0);
                #pragma unroll
                for (int tr = 0; tr < TR; ++tr) { const int r = tid + SW_CONSUMERS * tr; if (r < N) Y[r] = accY[0][tr]; }
            }
            consumer_sync();
            // y_P -= K y_T
            {
                cplx accK[SW_TCOLS];
                k_times(Y, accK, qT0, qT1);
                if (NC > 1) exchange(accK, SW_TCOLS, NP, Kpart, 1);
                #pragma unroll
                for (int tc = 0; tc < SW_TCOLS; ++tc) { const int r = tid + SW_CONSUMERS * tc; if (r < NP) { Y[NT + r].x -= accK[tc].x; Y[NT + r].y -= accK[tc].y; } }
            }
            consumer_sync();
            if (!SOLVE) {
                // w_P = Ainv y_P
                for (int q = 0; q < S.nA; ++q) {
                    const cplx *buf = acquire();
                    const int r0 = q * S.rA, rows = min(S.rA, NP - r0);
                    for (int r = warp; r < rows; r += 8) {
                        const cplx d = warp_dot(buf + (size_t)r * NP, Y + NT, NP, lane);
                        if (lane == 0) Wp[r0 + r] = d;
                    }
                    release();
                }
                consumer_sync();
            } else {
                // forward solve L w = y_P:  w_j = Linv_jj (y_j - sum_{i<j} L_ji w_i)
                for (int j = 0; j < CL.nblk; ++j) {
                    const int nbj = CL.nb(j), len = CL.len(j), j0 = CHOL_NB * j, rf = S.rows_fwd(CL, j);
                    for (int q0 = 0; q0 < nbj; q0 += rf) {
                        const cplx *buf = acquire();
                        const int rows = min(rf, nbj - q0);
                        for (int r = warp; r < rows; r += 8) {
                            const cplx *row = buf + (size_t)r * len;
                            const cplx d = warp_dot(row, Wp, j0, lane);
                            if (lane == 0) { const cplx y = Y[NT + j0 + q0 + r]; Tj[q0 + r] = {y.x - d.x, y.y - d.y}; }
                            if (lane < nbj) Dblk[(q0 + r) * SW_DLD + lane] = row[j0 + lane];
                        }
                        release();
                    }
                    consumer_sync();
                    for (int r = warp; r < nbj; r += 8) {
                        double sr = 0.0, si = 0.0;
                        if (lane <= r) { const cplx l = Dblk[r * SW_DLD + lane], x = Tj[lane]; sr = l.x * x.x - l.y * x.y; si = l.x * x.y + l.y * x.x; }
                        sr = warp_sum(sr); si = warp_sum(si);
                        if (lane == 0) Wp[j0 + r] = {sr, si};
                    }
                    consumer_sync();
                }
                // backward solve L^H x = w:  x_j = Linv_jj^H (w_j - sum_{i>j} L_ij^H x_i), in place in Wp
                for (int j = CL.nblk - 1; j >= 0; --j) {
                    const int nbj = CL.nb(j), j0 = CHOL_NB * j, below = NP - j0 - nbj, rb = S.rows_bwd(CL, j);
                    double pr = 0.0, pi = 0.0;                                   // lane = column c of block j
                    for (int q0 = 0; q0 < below; q0 += rb) {
                        const cplx *buf = acquire();
                        const int rows = min(rb, below - q0);
                        if (lane < nbj)
                            for (int r = warp; r < rows; r += 8) {
                                const cplx l = buf[(size_t)r * nbj + lane], x = Wp[j0 + nbj + q0 + r];
                                pr += l.x * x.x + l.y * x.y; pi += l.x * x.y - l.y * x.x;      // conj(l) x
                            }
                        release();
                    }
                    part2[warp * CHOL_NB + lane] = {pr, pi};
                    consumer_sync();
                    {
                        const cplx *buf = acquire();                            // Linv_jj [nbj][nbj]
                        if (warp == 0) {
                            if (lane < nbj) {
                                cplx u = Wp[j0 + lane];
                                for (int w = 0; w < 8; ++w) { u.x -= part2[w * CHOL_NB + lane].x; u.y -= part2[w * CHOL_NB + lane].y; }
                                Tj[lane] = u;
                            }
                            __syncwarp();
                            if (lane < nbj) {
                                double sr = 0.0, si = 0.0;
                                for (int k = lane; k < nbj; ++k) { const cplx l = buf[(size_t)k * nbj + lane], u = Tj[k]; sr += l.x * u.x + l.y * u.y; si += l.x * u.y - l.y * u.x; }
                                Wp[j0 + lane] = {sr, si};
                            }
                        }
                        release();
                    }
                    consumer_sync();
                }
            }
            // w_T = y_T - K^H w_P: thread c owns the columns c, c + 256, .. of K (consecutive lanes, conflict-free), reads
            // w_P[r] as a broadcast and accumulates over the streamed rows in registers: no partial sums, no reduction
            cplx accT[SW_TCOLS];
            #pragma unroll
            for (int tc = 0; tc < SW_TCOLS; ++tc) accT[tc] = cplx{0.0, 0.0};
            for (int q = qK0; q < qK1; ++q) {
                const cplx *buf = acquire();
                const int r0 = q * S.rK, rows = min(S.rK, NP - r0);
                for (int r = 0; r < rows; ++r) {
                    const cplx x = Wp[r0 + r];
                    const cplx *Kr = buf + (size_t)r * NT;
                    #pragma unroll
                    for (int tc = 0; tc < SW_TCOLS; ++tc) {
                        const int c = tid + SW_CONSUMERS * tc;
                        if (c < NT) { const cplx k = Kr[c]; accT[tc].x += k.x * x.x + k.y * x.y; accT[tc].y += k.x * x.y - k.y * x.x; }
                    }
                }
                release();
            }
            if (NC > 1) exchange(accT, SW_TCOLS, NT, Tpart, 2);
            // k = -(i/v) P w
            #pragma unroll
            for (int tr = 0; tr < TR; ++tr) {
                const int j = tid + SW_CONSUMERS * tr;
                if (j >= N) continue;
                cplx w;
                if (j < NT) {                                   // the column sums of K^H w_P for j = tid + 256 tr are this thread's own
                    w = Y[j];
                    if (tr < SW_TCOLS) { w.x -= accT[tr < SW_TCOLS ? tr : 0].x; w.y -= accT[tr < SW_TCOLS ? tr : 0].y; }
                } else w = Wp[j - NT];
                const cplx y = cmul(w, ph[tr]);
                const cplx k = {y.y / vel, -y.x / vel};
                Kn[tr] = k; Acc[tr].x += wgt * k.x; Acc[tr].y += wgt * k.y;
                if (st == 3) { C[tr].x += (h / 6.0) * Acc[tr].x; C[tr].y += (h / 6.0) * Acc[tr].y; Acc[tr] = cplx{0.0, 0.0}; Kn[tr] = cplx{0.0, 0.0}; }
            }
            consumer_sync();
        }
    }
    // a trajectory that met a failed factorisation (or had met one in an earlier window) has no amplitudes: NaN, and the
    // first failed half-step index is kept in traj_status (wpccc_last_status)
    const bool dead = first_bad < a.n_idx || (a.traj_status && a.traj_status[t] != 0);
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    if (NC > 1) cluster_sync_all();                  // neither CTA leaves (nor rank 0 touches traj_status) while the other may still read
    if (rank == 0) {
        #pragma unroll
        for (int tr = 0; tr < TR; ++tr) {
            const int j = tid + SW_CONSUMERS * tr;
            if (j < N) { double *dst = a.C + ((size_t)t * N + j) * 2; dst[0] = dead ? qnan : C[tr].x; dst[1] = dead ? qnan : C[tr].y; }
        }
        if (tid == 0 && a.traj_status && a.traj_status[t] == 0 && first_bad < a.n_idx)
            a.traj_status[t] = (a.flags[(size_t)t * a.n_idx + first_bad] << 28) | ((int)(a.i0 + first_bad) + 1);
        if (track && tid == 0) a.drift[t] = dead ? qnan : drift;
    }
}
}  // namespace

// (rows per thread, trajectories per unit) of the one-centre sweep for N states: 224 NTILE >= N, state in registers
static bool sweep1_shape(int N, int *ntile, int *nv) {
    static const int shapes[][3] = {{224, 1, 4}, {448, 2, 4}, {672, 3, 3}, {896, 4, 2}, {1344, 6, 1}, {2016, 9, 1}, {3136, 14, 1}, {4480, 20, 1}};
    for (auto &sh : shapes) if (N <= sh[0]) { *ntile = sh[1]; *nv = sh[2]; return true; }
    return false;
}
// kernel instance for units of at most `nmax` trajectories: the smallest NV >= nmax that is instantiated for this NTILE
static int sweep1_nv_instance(int ntile, int nv_plan, int nmax) {
    if (ntile <= 3 && nmax <= 1) return 1;
    if (ntile <= 2 && nmax <= 2) return 2;
    return nv_plan;
}

void wp_sweep1_plan(int N, int n_rad, int *nv, int *rows_per_chunk, int *stages) {
    (void)n_rad;
    int ntile = 1;
    if (!sweep1_shape(N, &ntile, nv)) { *nv = 1; *rows_per_chunk = 1; *stages = 2; return; }      // wp_sweep_one_centre reports the limit
    // ring of whole rows + the double-buffered stage vectors within the 227 KB of a CTA.  One SM's TMA bulk-copy stream
    // delivers about chunk / 0.36 us whatever the ring depth (measured: 16 KB chunks 46 GB/s, 32 KB 88, 48 KB 107, 64 KB 133 GB/s):
    // three stages of up to 56 KB
    const int ld = wp_sweep1_ld(N);
    const size_t cap = 220 * 1024, vec = (size_t)2 * *nv * N * 16;
    int rr = std::max(1, std::min(64, (int)(57344 / ((size_t)ld * 8)))), ss = 3;
    while (rr > 1 && (size_t)ss * rr * ld * 8 + vec > cap) --rr;
    while (ss > 2 && (size_t)ss * rr * ld * 8 + vec > cap) --ss;
    *rows_per_chunk = rr; *stages = ss;
}

int wp_sweep_one_centre(wpccc_basis *B, int n_units, const Sweep1Args &a_in, cudaStream_t s) {
    if (n_units <= 0 || a_in.steps <= 0) return 0;
    Sweep1Args a = a_in;
    int ntile = 0, nvs = 0;
    if (!sweep1_shape(a.N, &ntile, &nvs)) WP_FAIL(WPCCC_EINVAL, "one-centre sweep: N = %d exceeds the register-resident design (N <= 4480)", a.N);
    const int nvi = sweep1_nv_instance(ntile, nvs, a.nv);           // a.nv: largest unit of this call
    // a cluster of two CTAs per unit when the units leave more than half of the SMs idle and a stage is bound by one SM's streams
    int nc = (a.N >= 384 && ntile >= 2 && ntile <= 4 && 2 * n_units <= 148) ? 2 : 1;
    if (B->opt.sweep_cluster == 1) nc = 1;
    else if (B->opt.sweep_cluster >= 2 && ntile >= 2 && ntile <= 4) nc = 2;
    const size_t vec = (size_t)2 * nvi * a.N * 16, part = (size_t)nvi * a.N * 16;
    static PerDevice attr_1;
    const bool raise = wp_raise(attr_1, 1);               // once per device: every instance gets the full shared-memory limit
    wp_span_begin(B, FAM_SWEEP, s);
#define WP_SWEEP1C(NT_, NV_, NC_) do { static PerDevice at_; if (raise || wp_raise(at_, 1)) WP_CUDA(cudaFuncSetAttribute(k_sweep1<NT_, NV_, NC_>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024)); \
        lerr = cudaLaunchKernelEx(&lc, k_sweep1<NT_, NV_, NC_>, a); } while (0)
#define WP_SWEEP1(NT_, NV_) WP_SWEEP1C(NT_, NV_, 1)
#define WP_SWEEP1X(NT_, NV_) do { if (nc > 1) WP_SWEEP1C(NT_, NV_, 2); else WP_SWEEP1C(NT_, NV_, 1); } while (0)
    for (;;) {
        a.rows_per_chunk = a_in.rows_per_chunk;
        if (nc > 1) {                                        // room for the partial sums: shorter chunks
            while (a.rows_per_chunk > 1 && (size_t)a.ring_stages * a.rows_per_chunk * a.ldD * 8 + vec + part > 225 * 1024) --a.rows_per_chunk;
            if ((size_t)a.ring_stages * a.rows_per_chunk * a.ldD * 8 + vec + part > 225 * 1024) { nc = 1; a.rows_per_chunk = a_in.rows_per_chunk; }
        }
        const size_t smem = (size_t)a.ring_stages * a.rows_per_chunk * a.ldD * 8 + vec + (nc > 1 ? part : 0);
        if (smem > 227 * 1024 - 1024) WP_FAIL(WPCCC_EINVAL, "one-centre sweep: N = %d too large for shared memory", a.N);
        cudaLaunchConfig_t lc{};
        cudaLaunchAttribute lattr[1];
        lc.gridDim = dim3((unsigned)(n_units * nc)); lc.blockDim = dim3(SW1_CONSUMERS + 32); lc.dynamicSmemBytes = smem; lc.stream = s;
        lattr[0].id = cudaLaunchAttributeClusterDimension; lattr[0].val.clusterDim.x = (unsigned)nc; lattr[0].val.clusterDim.y = 1; lattr[0].val.clusterDim.z = 1;
        lc.attrs = lattr; lc.numAttrs = 1;
        cudaError_t lerr = cudaSuccess;
        switch (ntile) {
            case 1: if (nvi == 1) WP_SWEEP1(1, 1); else if (nvi == 2) WP_SWEEP1(1, 2); else WP_SWEEP1(1, 4); break;
            case 2: if (nvi == 1) WP_SWEEP1X(2, 1); else if (nvi == 2) WP_SWEEP1X(2, 2); else WP_SWEEP1X(2, 4); break;
            case 3: if (nvi == 1) WP_SWEEP1X(3, 1); else WP_SWEEP1X(3, 3); break;
            case 4: WP_SWEEP1X(4, 2); break;
            case 6: WP_SWEEP1(6, 1); break;
            case 9: WP_SWEEP1(9, 1); break;
            case 14: WP_SWEEP1(14, 1); break;
            default: WP_SWEEP1(20, 1); break;
        }
        if (lerr == cudaSuccess) break;
        (void)cudaGetLastError();
        if (nc == 1) { wp_set_error("one-centre sweep: launch failed -> %s", cudaGetErrorString(lerr)); return WPCCC_ECUDA; }
        nc = 1;                                          // the cluster cannot be placed on this device: one CTA per unit
    }
#undef WP_SWEEP1
#undef WP_SWEEP1X
#undef WP_SWEEP1C
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}

int wp_sweep_two_centre(wpccc_basis *B, int n_traj, const Sweep2Args &a, cudaStream_t s) {
    if (n_traj <= 0 || a.steps <= 0) return 0;
    const int N = a.NT + a.NP;
    if (a.NT > SW_CONSUMERS * SW_TCOLS || a.NP > SW_CONSUMERS * SW_TCOLS) WP_FAIL(WPCCC_EINVAL, "two-centre sweep: N_T = %d or N_P = %d exceeds %d", a.NT, a.NP, SW_CONSUMERS * SW_TCOLS);
    if (N > SW_CONSUMERS * 8) WP_FAIL(WPCCC_EINVAL, "two-centre sweep: N = %d exceeds %d", N, SW_CONSUMERS * 8);
    // a cluster of CTAs per trajectory: the streams of one SM bound a stage of a wide basis, and even at N = 172 halving them pays
    const int tr = (N + SW_CONSUMERS - 1) / SW_CONSUMERS;
    int cl = (N >= 512) ? 4 : ((N >= 128) ? 2 : 1);     // measured: configs[1] (N = 172) 229 -> 164 ms of sweep per job with two CTAs (154 with four, but
                                                        // the element stream then loses more than that); configs[3] (N = 572) 1.77 -> 1.40 -> 1.06 s
    if (B->opt.sweep_cluster) cl = B->opt.sweep_cluster;
    // kernel instances: one CTA for TR <= 2, two CTAs for TR <= 2, four CTAs for any TR
    if (cl == 1 && tr > 2) cl = 2;
    if (cl == 2 && tr > 2) cl = 4;
    wp_span_begin(B, FAM_SWEEP, s);
#define WP_SWEEP2(SOLVE_, TR_, NC_) do { static PerDevice at_; if (wp_raise(at_, 1)) WP_CUDA(cudaFuncSetAttribute(k_sweep2<SOLVE_, TR_, NC_>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024)); \
        lerr = cudaLaunchKernelEx(&lc, k_sweep2<SOLVE_, TR_, NC_>, a, chunk_i, NS); } while (0)
#define WP_SWEEP2_TR(SOLVE_) do { if (cl == 1) { if (tr <= 1) WP_SWEEP2(SOLVE_, 1, 1); else WP_SWEEP2(SOLVE_, 2, 1); } \
        else if (cl == 2) WP_SWEEP2(SOLVE_, 2, 2); \
        else if (tr <= 3) WP_SWEEP2(SOLVE_, 3, 4); else if (tr == 4) WP_SWEEP2(SOLVE_, 4, 4); else WP_SWEEP2(SOLVE_, 8, 4); } while (0)
    for (;;) {
        const size_t vec = ((size_t)2 * N + a.NP + CHOL_NB + CHOL_NB * SW_DLD + 8 * CHOL_NB + (cl > 1 ? 2 * (size_t)N : 0)) * 16;
        // TMA ring: one SM's bulk-copy stream delivers about chunk / 0.36 us whatever the ring depth (measured: 16 KB chunks 46 GB/s,
        // 32 KB 88, 48 KB 107, 64 KB 133 GB/s), so the chunks are as large as the shared memory allows: three stages of up to 64 KB,
        // two stages when three would be smaller than 48 KB each
        const size_t chunk_min = std::max((size_t)16 * N, (size_t)16 * CHOL_NB * CHOL_NB), room = (size_t)220 * 1024 - vec;
        int NS = 3;
        size_t chunk = std::min<size_t>(64 * 1024, room / 3);
        if (chunk < 48 * 1024) { NS = 2; chunk = std::min<size_t>(96 * 1024, room / 2); }
        chunk &= ~(size_t)127;
        if (chunk < chunk_min) WP_FAIL(WPCCC_EINVAL, "two-centre sweep: N = %d too large for shared memory", N);
        const size_t smem = NS * chunk + vec;
        if (smem > 225 * 1024) WP_FAIL(WPCCC_EINVAL, "two-centre sweep: N = %d too large for shared memory", N);
        cudaLaunchConfig_t lc{};
        cudaLaunchAttribute lattr[1];
        lc.gridDim = dim3((unsigned)(n_traj * cl)); lc.blockDim = dim3(SW_CONSUMERS + 32); lc.dynamicSmemBytes = smem; lc.stream = s;
        lattr[0].id = cudaLaunchAttributeClusterDimension; lattr[0].val.clusterDim.x = (unsigned)cl; lattr[0].val.clusterDim.y = 1; lattr[0].val.clusterDim.z = 1;
        lc.attrs = lattr; lc.numAttrs = 1;
        const int chunk_i = (int)chunk;
        cudaError_t lerr = cudaSuccess;
        if (a.solve) WP_SWEEP2_TR(true); else WP_SWEEP2_TR(false);
        if (lerr == cudaSuccess) break;
        (void)cudaGetLastError();
        // a cluster of this size cannot be placed on this device (fewer SMs per GPC, a partitioned GPU): the next smaller size
        // that has a kernel instance for this basis, if any
        if (cl == 1 || tr > 2) { wp_set_error("two-centre sweep: launch failed with %d CTAs per trajectory -> %s", cl, cudaGetErrorString(lerr)); return WPCCC_ECUDA; }
        cl /= 2;
    }
#undef WP_SWEEP2_TR
#undef WP_SWEEP2
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}

int wp_factor_cholesky(wpccc_basis *B, int n_pos, const double *d_K, double *d_out, int *d_flags, void *d_scratch, cudaStream_t s);

int wp_factor(wpccc_basis *B, int n_pos, const double *d_K, double *d_Ainv, int *d_flags, void *d_scratch, cudaStream_t s) {
    if (n_pos <= 0) return 0;
    if (B->opt.solve_route == 0) return wp_factor_cholesky(B, n_pos, d_K, d_Ainv, d_flags, d_scratch, s);
    FactorArgs a{};
    a.K = d_K; a.Ainv = d_Ainv; a.flags = d_flags; a.NT = B->c[0].n_states; a.NP = B->c[1].n_states; a.out_stride = wp_factor_elems(a.NP);
    const size_t n = a.NP, small = 2 * n * 16 + 2 * n * 4 + 64;
    const size_t budget = 200 * 1024;
    const bool force_blocked = B->opt.inverse_kernel == 2;                   // wpccc_set_option "inverse_kernel": global-memory blocked route
    const bool no_reg = B->opt.inverse_kernel == 1;                          // shared-memory route
    if (n <= (size_t)FR_NMAX && !force_blocked && !no_reg) {                    // A in registers
        const size_t tail = (2 * FR_NMAX * FR_NB + FR_NB * FR_NMAX) * 16 + 4 * FR_NMAX * 4;
        size_t cwr = (size_t)a.NT | 1;                                        // odd row stride: conflict-free column reads
        const size_t cw_max = ((160 * 1024 - tail) / (n * 16) - 1) | 1;
        if (cwr > cw_max) cwr = cw_max;
        if (B->opt.inverse_chunk_cols > 0) { const size_t t = (size_t)B->opt.inverse_chunk_cols | 1; if (t < cwr) cwr = t; }   // K staged in several chunks
        a.cw = (int)cwr;
        const size_t smem = n * cwr * 16 + tail;
        static PerDevice attr_r;
        if (wp_raise(attr_r, smem)) WP_CUDA(cudaFuncSetAttribute(k_factor_reg, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        wp_span_begin(B, FAM_FACT, s);
        k_factor_reg<<<n_pos, FR_THREADS, smem, s>>>(a);
        wp_span_end(B, s, 1);
        WP_CUDA(cudaGetLastError());
        return 0;
    }
    a.use_smem = !force_blocked && n * n * 16 + n * (2 * FJ_NB + 1) * 16 + small <= budget;   // K chunk area doubles as the panel buffers
    const size_t fixed = (a.use_smem ? n * n * 16 : 0) + small;
    // large N_P (blocked path): two CTAs per SM; the K staging area is reused by the panel buffers (2 FJ_NB + 1 columns)
    const size_t blocked_need = (2 * FJ_NB + 1) * n * 16 + n * 4 + 64;
    const size_t kbudget = a.use_smem ? budget : std::max<size_t>(blocked_need, 100 * 1024);
    if (!a.use_smem && blocked_need > budget) WP_FAIL(WPCCC_EINVAL, "factorisation: N_P = %d too large", a.NP);
    int cw = (int)std::min<size_t>((kbudget - fixed) / (n * 16), (size_t)a.NT);
    if (cw > 1 && (cw & 1) == 0) --cw;                        // odd width: conflict-free column reads
    if (cw < 1) WP_FAIL(WPCCC_EINVAL, "factorisation: N_P = %d too large", a.NP);
    if (a.use_smem && cw < 2 * FJ_NB + 1) cw = 2 * FJ_NB + 1;    // the K chunk area doubles as the panel buffers (N_T < 17)
    a.cw = cw;
    const size_t smem = a.use_smem ? fixed + n * cw * 16 : std::max(fixed + n * cw * 16, blocked_need);
    static PerDevice attr_f;
    if (wp_raise(attr_f, smem)) WP_CUDA(cudaFuncSetAttribute(k_factor, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    wp_span_begin(B, FAM_FACT, s);
    k_factor<<<n_pos, 512, smem, s>>>(a);
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}
