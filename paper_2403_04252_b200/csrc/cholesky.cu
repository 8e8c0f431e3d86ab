// a7, solve route 0 (wpccc_set_option "solve_route"): the overlap system S = [[I, K^H], [K, I]] of eq. (4)
// is reduced to its Schur complement A = I - K K^H (Hermitian; positive definite exactly when S is), which is
// factorised A = L L^H by a blocked right-looking Cholesky algorithm, batched over the positions of a window:
//   k_herk<init>   A = I - K K^H, and the trailing updates A22 -= L21 L21^H, on the FP64 tensor cores (complex HERK as four
//                  real mma.sync.m8n8k4.f64 products per k4-step; lower-triangle tiles only);
//   k_chol_step    block step j: Cholesky of the 32 x 32 diagonal block and its triangular inverse by one warp in shared
//                  memory, then the panel L21 = A21 Linv_jj^H by all warps; writes the packed factor of sweep.cuh.
// The RK4 sweep then does two blocked triangular solves per stage (a linear solve, as PAPER.md L61 asks, not an inverse).
// A block whose pivot is not positive flags the position (3: not positive definite): with an over-complete two-centre
// basis the configured quadrature can leave S(R) indefinite at small R (A23).
#include "sweep.cuh"
#include "ptx.cuh"

namespace {

constexpr int HK_T = 32, HK_KC = 32, HK_LD = HK_KC + 4, HK_THREADS = 128;     // tile, k-chunk, padded row stride (complex), threads

struct HerkArgs {
    const cplx *P; cplx *C;            // per position: P [m][ldp] (kdim columns used), C [m][ldc]
    size_t p_stride, c_stride;         // complex elements between positions
    int m, kdim, ldp, ldc;
};

// grid = (lower tiles of the m x m result, positions); 4 warps, warp tile 16 x 16 complex of a 32 x 32 tile.
// INIT: C = I - P P^H, else C -= P P^H.  Only elements with row >= col are stored.
template <bool INIT>
__global__ void __launch_bounds__(HK_THREADS) k_herk(const HerkArgs a) {
    extern __shared__ __align__(16) unsigned char hk_raw[];
    cplx *sm = reinterpret_cast<cplx *>(hk_raw);                 // [2 stages][2 operands][HK_T][HK_LD]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int ti = (int)((sqrtf(8.0f * (float)blockIdx.x + 1.0f) - 1.0f) * 0.5f);
    while ((ti + 1) * (ti + 2) / 2 <= (int)blockIdx.x) ++ti;
    while (ti * (ti + 1) / 2 > (int)blockIdx.x) --ti;
    const int tj = (int)blockIdx.x - ti * (ti + 1) / 2;
    const cplx *P = a.P + (size_t)blockIdx.y * a.p_stride;
    cplx *C = a.C + (size_t)blockIdx.y * a.c_stride;
    const int r0 = ti * HK_T, c0 = tj * HK_T, nch = (a.kdim + HK_KC - 1) / HK_KC;

    auto load = [&](int stage, int ch) {
        cplx *dA = sm + (size_t)stage * 2 * HK_T * HK_LD, *dB = dA + HK_T * HK_LD;
        const int k0 = ch * HK_KC;
        #pragma unroll
        for (int it = 0; it < (HK_T * HK_KC) / HK_THREADS; ++it) {
            const int e = tid + it * HK_THREADS, r = e / HK_KC, q = e % HK_KC;
            const bool kin = k0 + q < a.kdim;
            if (kin && r0 + r < a.m) cp_async16(dA + r * HK_LD + q, P + (size_t)(r0 + r) * a.ldp + k0 + q); else dA[r * HK_LD + q] = cplx{0.0, 0.0};
            if (kin && c0 + r < a.m) cp_async16(dB + r * HK_LD + q, P + (size_t)(c0 + r) * a.ldp + k0 + q); else dB[r * HK_LD + q] = cplx{0.0, 0.0};
        }
        cp_async_commit();
    };
    double Cre[2][2][2], Cim[2][2][2];
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < 2; ++j) { Cre[i][j][0] = Cre[i][j][1] = Cim[i][j][0] = Cim[i][j][1] = 0.0; }
    const int wr = warp >> 1, wc = warp & 1, fr = lane >> 2, fk = lane & 3;
    load(0, 0);
    for (int ch = 0; ch < nch; ++ch) {
        if (ch + 1 < nch) { load((ch + 1) & 1, ch + 1); cp_async_wait<1>(); } else cp_async_wait<0>();
        __syncthreads();
        const cplx *sA = sm + (size_t)(ch & 1) * 2 * HK_T * HK_LD + (16 * wr + fr) * HK_LD + fk;
        const cplx *sB = sm + (size_t)(ch & 1) * 2 * HK_T * HK_LD + HK_T * HK_LD + (16 * wc + fr) * HK_LD + fk;
        #pragma unroll
        for (int k4 = 0; k4 < HK_KC / 4; ++k4) {
            cplx av[2], bv[2];
            #pragma unroll
            for (int i = 0; i < 2; ++i) { av[i] = sA[8 * i * HK_LD + 4 * k4]; bv[i] = sB[8 * i * HK_LD + 4 * k4]; }
            #pragma unroll
            for (int i = 0; i < 2; ++i)
                #pragma unroll
                for (int j = 0; j < 2; ++j) {
                    // (a.x + i a.y) conj(b.x + i b.y) = a.x b.x + a.y b.y + i (a.y b.x - a.x b.y)
                    dmma884(Cre[i][j][0], Cre[i][j][1], av[i].x, bv[j].x);
                    dmma884(Cre[i][j][0], Cre[i][j][1], av[i].y, bv[j].y);
                    dmma884(Cim[i][j][0], Cim[i][j][1], av[i].y, bv[j].x);
                    dmma884(Cim[i][j][0], Cim[i][j][1], -av[i].x, bv[j].y);
                }
        }
        __syncthreads();
    }
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < 2; ++j)
            #pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int row = r0 + 16 * wr + 8 * i + fr, col = c0 + 16 * wc + 8 * j + 2 * fk + e;
                if (row < a.m && col <= row) {
                    cplx *dst = C + (size_t)row * a.ldc + col;
                    cplx old = INIT ? cplx{row == col ? 1.0 : 0.0, 0.0} : *dst;
                    *dst = cplx{old.x - Cre[i][j][e], old.y - Cim[i][j][e]};
                }
            }
}

struct CholStepArgs {
    cplx *A; size_t a_stride;           // scratch: the (partially updated) Schur complement, [n][n] per position
    cplx *out; size_t out_stride;       // packed factor (CholLayout), per position
    int *flags;
    int n, j;                           // block step
};

constexpr int CS_LD = CHOL_NB + 1, CS_THREADS = 256;

// grid = positions; block = 8 warps.
__global__ void __launch_bounds__(CS_THREADS) k_chol_step(const CholStepArgs a) {
    __shared__ cplx D[CHOL_NB * CS_LD], Li[CHOL_NB * CS_LD];
    __shared__ int s_bad;
    const CholLayout L(a.n);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, j = a.j, nbj = L.nb(j), j0 = CHOL_NB * j, n = a.n;
    cplx *A = a.A + (size_t)blockIdx.x * a.a_stride;
    cplx *out = a.out + (size_t)blockIdx.x * a.out_stride;
    if (tid == 0) s_bad = 0;
    for (int e = tid; e < CHOL_NB * CHOL_NB; e += CS_THREADS) {
        const int r = e / CHOL_NB, c = e % CHOL_NB;
        D[r * CS_LD + c] = (r < nbj && c <= r) ? A[(size_t)(j0 + r) * n + j0 + c] : cplx{0.0, 0.0};
        Li[r * CS_LD + c] = cplx{0.0, 0.0};
    }
    __syncthreads();
    if (warp == 0) {
        // Cholesky of the diagonal block, lane = row: column k is scaled by 1 / sqrt(pivot), then the rows below are updated
        int bad = 0;
        for (int k = 0; k < nbj; ++k) {
            __syncwarp();                                                  // the updates of step k - 1 are visible
            const double d2 = D[k * CS_LD + k].x;
            if (!(d2 > 0.0) || !(d2 < 1.0e300)) bad = 1;                  // not positive definite (or not finite)
            const double d = sqrt(d2), inv = 1.0 / d;
            __syncwarp();
            if (lane == k) D[k * CS_LD + k] = cplx{d, 0.0};
            else if (lane > k && lane < nbj) { cplx x = D[lane * CS_LD + k]; D[lane * CS_LD + k] = cplx{x.x * inv, x.y * inv}; }
            __syncwarp();
            if (lane > k && lane < nbj) {
                const cplx lk = D[lane * CS_LD + k];
                for (int c = k + 1; c <= lane; ++c) {
                    const cplx lc = D[c * CS_LD + k];
                    cplx x = D[lane * CS_LD + c];
                    x.x -= lk.x * lc.x + lk.y * lc.y; x.y -= lk.y * lc.x - lk.x * lc.y;        // lk conj(lc)
                    D[lane * CS_LD + c] = x;
                }
            }
        }
        if (bad && lane == 0) s_bad = 1;
        __syncwarp();
        // inverse of the lower-triangular block, lane = column c: forward substitution L x = e_c
        if (lane < nbj) {
            const int c = lane;
            Li[c * CS_LD + c] = cplx{1.0 / D[c * CS_LD + c].x, 0.0};
            for (int r = c + 1; r < nbj; ++r) {
                double sr = 0.0, si = 0.0;
                for (int k = c; k < r; ++k) { const cplx l = D[r * CS_LD + k], x = Li[k * CS_LD + c]; sr += l.x * x.x - l.y * x.y; si += l.x * x.y + l.y * x.x; }
                const double inv = 1.0 / D[r * CS_LD + r].x;
                Li[r * CS_LD + c] = cplx{-sr * inv, -si * inv};
            }
        }
    }
    __syncthreads();
    if (tid == 0 && s_bad) a.flags[blockIdx.x] = 3;
    // the inverse of the diagonal block goes into both packed copies
    {
        cplx *dr = out + L.off_r(j), *dc = out + L.off_c(j);
        const int len = L.len(j);
        for (int e = tid; e < nbj * nbj; e += CS_THREADS) {
            const int r = e / nbj, c = e % nbj;
            const cplx v = Li[r * CS_LD + c];
            dr[(size_t)r * len + j0 + c] = v; dc[(size_t)r * nbj + c] = v;
        }
    }
    // panel: L21 = A21 Linv_jj^H, one warp per row r below the block: out[c] = sum_{k <= c} A[r][j0 + k] conj(Linv[c][k])
    if (j + 1 < L.nblk) {
        cplx *dc = out + L.off_c(j);
        for (int r = j0 + CHOL_NB + warp; r < n; r += CS_THREADS / 32) {
            const cplx av = A[(size_t)r * n + j0 + lane];
            double sr = 0.0, si = 0.0;
            #pragma unroll 8
            for (int k = 0; k < CHOL_NB; ++k) {
                const double ax = __shfl_sync(0xffffffffu, av.x, k), ay = __shfl_sync(0xffffffffu, av.y, k);
                const cplx li = Li[lane * CS_LD + k];                          // zero for k > lane
                sr += ax * li.x + ay * li.y; si += ay * li.x - ax * li.y;
            }
            const cplx v = {sr, si};
            A[(size_t)r * n + j0 + lane] = v;
            dc[(size_t)(r - j0) * CHOL_NB + lane] = v;
            const int jr = r / CHOL_NB;
            out[L.off_r(jr) + (size_t)(r - CHOL_NB * jr) * L.len(jr) + j0 + lane] = v;
        }
    }
}

}  // namespace

size_t wp_factor_scratch_bytes(const wpccc_basis *B, int n_pos) {
    if (B->n_centres != 2) return 0;
    const size_t n = B->c[1].n_states;
    return (size_t)n_pos * n * n * 16 + 256;
}

int wp_factor_cholesky(wpccc_basis *B, int n_pos, const double *d_K, double *d_out, int *d_flags, void *d_scratch, cudaStream_t s) {
    if (n_pos <= 0) return 0;
    const int NT = B->c[0].n_states, n = B->c[1].n_states;
    const CholLayout L(n);
    cplx *A = reinterpret_cast<cplx *>(d_scratch);
    const size_t smem = (size_t)2 * 2 * HK_T * HK_LD * sizeof(cplx);
    static PerDevice attr;
    if (wp_raise(attr, smem)) {
        WP_CUDA(cudaFuncSetAttribute(k_herk<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        WP_CUDA(cudaFuncSetAttribute(k_herk<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    }
    wp_span_begin(B, FAM_FACT, s);
    int launches = 0;
    for (int p0 = 0; p0 < n_pos; p0 += 32768) {                        // grid.y limit
        const int np = std::min(32768, n_pos - p0);
        HerkArgs h{};
        h.P = reinterpret_cast<const cplx *>(d_K) + (size_t)p0 * n * NT; h.p_stride = (size_t)n * NT; h.ldp = NT; h.kdim = NT;
        h.C = A + (size_t)p0 * n * n; h.c_stride = (size_t)n * n; h.ldc = n; h.m = n;
        const int mt = (n + HK_T - 1) / HK_T;
        k_herk<true><<<dim3(mt * (mt + 1) / 2, np), HK_THREADS, smem, s>>>(h);
        ++launches;
        for (int j = 0; j < L.nblk; ++j) {
            CholStepArgs c{};
            c.A = A + (size_t)p0 * n * n; c.a_stride = (size_t)n * n; c.out = reinterpret_cast<cplx *>(d_out) + (size_t)p0 * wp_factor_elems(n);
            c.out_stride = wp_factor_elems(n); c.flags = d_flags + p0; c.n = n; c.j = j;
            k_chol_step<<<np, CS_THREADS, 0, s>>>(c);
            ++launches;
            const int m = n - CHOL_NB * (j + 1);
            if (m > 0) {
                HerkArgs t{};
                t.P = A + (size_t)p0 * n * n + (size_t)CHOL_NB * (j + 1) * n + CHOL_NB * j; t.p_stride = (size_t)n * n; t.ldp = n; t.kdim = CHOL_NB;
                t.C = A + (size_t)p0 * n * n + (size_t)CHOL_NB * (j + 1) * (n + 1); t.c_stride = (size_t)n * n; t.ldc = n; t.m = m;
                const int mt2 = (m + HK_T - 1) / HK_T;
                k_herk<false><<<dim3(mt2 * (mt2 + 1) / 2, np), HK_THREADS, smem, s>>>(t);
                ++launches;
            }
        }
    }
    wp_span_end(B, s, launches);
    WP_CUDA(cudaGetLastError());
    return 0;
}
