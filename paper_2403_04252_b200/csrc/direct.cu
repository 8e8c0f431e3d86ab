// Direct (one-centre) couplings: eq. (6)-(7) of the paper.
//
// a2  radial contraction  F^c_lambda(a',a;R_p) = sum_k V_lambda(r_k,R_p) * PP[(a',a)][k],
//     PP[(a',a)][k] = w_k u_a'(r_k) u_a(r_k),  V_lambda(r,R) = min(r,R)^lambda / max(r,R)^(lambda+1)
//     as a grouped FP64 tensor-core GEMM (mma.sync m8n8k4 = SASS DMMA.8x8x4): one group per multipole lambda,
//     M = positions, N = pairs allowed for lambda, K = radial grid.  The M operand V is generated on the fly
//     from the r^lambda / r^-(lambda+1) tables; the N operand streams from the pair-product matrix in HBM/L2
//     with cp.async double buffering.
// a3  assembly  D_{alpha' alpha} = -Z sum_lambda (+-1)^lambda G^lambda_{alpha' alpha} P_lambda^{m'-m}(cos Theta) F_lambda
#include <algorithm>

#include "common.cuh"
#include "ptx.cuh"

namespace {

constexpr int BM = 128, BN = 128, BK = 32, LDS_ = BK + 4;   // row stride 36 doubles: conflict-free fragment reads
constexpr int GEMM_THREADS = 256, NSTG = 3;    // three k-chunks in flight, one block-wide barrier per chunk


struct GemmArgs {
    const GemmTile *tiles;
    const double *PP[2];
    const int *ent_pair[2];
    int lam_off[2][WP_MAX_LAMBDA + 2];
    int cen_off[2];
    const double *rp, *rm, *rk;
    const double *R;
    double *F;
    int ldF, n_pos, Kpad;
    PosMap rmap, fmap;
};

// grid: (m tiles, n tiles).  256 threads = 8 warps as 2 (M) x 4 (N); warp tile 64 x 32 -> 32 DMMA per k4 step.
__global__ void __launch_bounds__(GEMM_THREADS, 1) k_direct_gemm(const GemmArgs a) {
    extern __shared__ __align__(16) double smem[];
    double *As = smem;                         // [NSTG][BM][LDS_]
    double *Bs = smem + NSTG * BM * LDS_;      // [NSTG][BN][LDS_]
    __shared__ double sR[BM], sRp[BM], sRm[BM];
    __shared__ int sPair[BN];

    const GemmTile t = a.tiles[blockIdx.y];
    const int m0 = blockIdx.x * BM;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lam = t.lam;

    if (tid < BM) {
        int p = m0 + tid;
        double R = (p < a.n_pos) ? a.R[pos_row(a.rmap, p)] : 1.0;
        double Rp = 1.0;
        for (int i = 0; i < lam; ++i) Rp *= R;
        sR[tid] = R; sRp[tid] = Rp; sRm[tid] = 1.0 / (Rp * R);
    }
    if (tid < BN) {
        int n = t.n0 + tid;
        sPair[tid] = (tid < t.cnt) ? a.ent_pair[t.c][a.lam_off[t.c][lam] + n] : -1;
    }
    __syncthreads();

    const double *PP = a.PP[t.c];
    const double *rp = a.rp + (size_t)lam * a.Kpad, *rm = a.rm + (size_t)lam * a.Kpad;
    const int nk = a.Kpad / BK;

    auto load_B = [&](int buf, int kc) {
        double *dst = Bs + buf * BN * LDS_;
        #pragma unroll
        for (int j = 0; j < (BN * BK / 2) / GEMM_THREADS; ++j) {
            int c = tid + GEMM_THREADS * j, row = c >> 4, part = c & 15;
            int pr = sPair[row];
            double *d = dst + row * LDS_ + part * 2;
            if (pr >= 0) cp_async16(d, PP + (size_t)pr * a.Kpad + kc * BK + part * 2);
            else { d[0] = 0.0; d[1] = 0.0; }
        }
    };
    auto gen_A = [&](int buf, int kc) {
        double *dst = As + buf * BM * LDS_;
        const int k = tid & 31, r0 = tid >> 5;
        const double rkk = a.rk[kc * BK + k], rpk = rp[kc * BK + k], rmk = rm[kc * BK + k];
        #pragma unroll
        for (int j = 0; j < BM / 8; ++j) {
            int row = r0 + 8 * j;
            dst[row * LDS_ + k] = (rkk < sR[row]) ? rpk * sRm[row] : rmk * sRp[row];
        }
    };

    double acc[8][4][2];
    #pragma unroll
    for (int i = 0; i < 8; ++i)
        #pragma unroll
        for (int j = 0; j < 4; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

    // warps w and w + 4 share an SM sub-partition: give them N offsets 64 apart, so that a ragged tile (cnt <= 64) leaves
    // one active warp on every sub-partition instead of two sub-partitions idle
    const int wm = (warp & 1) * 64, wn = (warp >> 1) * 32;
    const bool warp_active = (wn < t.cnt);
    const int fr = lane >> 2, fk = lane & 3;

    load_B(0, 0); cp_async_commit(); gen_A(0, 0);
    if (nk > 1) { load_B(1, 1); gen_A(1, 1); }
    cp_async_commit();
    for (int kc = 0; kc < nk; ++kc) {
        const int buf = kc % NSTG;
        cp_async_wait<1>();                    // this thread's copies of chunk kc have landed
        __syncthreads();                       // chunk kc complete for everyone; buffer of chunk kc - 1 is free again
        if (kc + 2 < nk) { load_B((kc + 2) % NSTG, kc + 2); gen_A((kc + 2) % NSTG, kc + 2); }
        cp_async_commit();
        if (warp_active) {
            const double *Ab = As + buf * BM * LDS_ + (wm + fr) * LDS_ + fk;
            const double *Bb = Bs + buf * BN * LDS_ + (wn + fr) * LDS_ + fk;
            #pragma unroll
            for (int ks = 0; ks < BK / 4; ++ks) {
                double af[8], bf[4];
                #pragma unroll
                for (int i = 0; i < 8; ++i) af[i] = Ab[i * 8 * LDS_ + ks * 4];
                #pragma unroll
                for (int j = 0; j < 4; ++j) bf[j] = Bb[j * 8 * LDS_ + ks * 4];
                #pragma unroll
                for (int i = 0; i < 8; ++i)
                    #pragma unroll
                    for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            }
        }
    }
    if (!warp_active) return;
    const int colbase = a.cen_off[t.c] + a.lam_off[t.c][lam] + t.n0;
    #pragma unroll
    for (int i = 0; i < 8; ++i) {
        int p = m0 + wm + 8 * i + fr;
        if (p >= a.n_pos) continue;
        double *Frow = a.F + pos_row(a.fmap, p) * a.ldF + colbase;
        #pragma unroll
        for (int j = 0; j < 4; ++j) {
            int n = wn + 8 * j + 2 * fk;
            if (n < t.cnt) Frow[n] = acc[i][j][0];
            if (n + 1 < t.cnt) Frow[n + 1] = acc[i][j][1];
        }
    }
}

// Associated Legendre functions P_lambda^mu(x), Condon-Shortley phase, all 0 <= lambda <= L, |mu| <= lambda,
// into P[lambda * ldp + mu + L].  One thread; L <= WP_MAX_LAMBDA.
__device__ void assoc_legendre_all(int L, double x, double *P, int ldp) {
    const double s = sqrt(fmax(0.0, 1.0 - x * x));
    double pmm = 1.0;
    for (int m = 0; m <= L; ++m) {
        if (m > 0) pmm = -pmm * (2 * m - 1) * s;
        double p0 = pmm, p1 = x * (2 * m + 1) * pmm;
        // factorial ratio (lambda-m)!/(lambda+m)! built incrementally
        for (int lam = m; lam <= L; ++lam) {
            double val;
            if (lam == m) val = p0;
            else if (lam == m + 1) val = p1;
            else { val = ((2 * lam - 1) * x * p1 - (lam + m - 1) * p0) / (lam - m); p0 = p1; p1 = val; }
            P[lam * ldp + m + L] = val;
            if (m > 0) {
                double ratio = 1.0;                      // (lam-m)!/(lam+m)!
                for (int q = lam - m + 1; q <= lam + m; ++q) ratio /= q;
                P[lam * ldp - m + L] = ((m & 1) ? -ratio : ratio) * val;
            }
        }
    }
}

struct AsmArgs {
    const double *G; const int *ent_lookup; const int *st_rad, *st_l, *st_m;
    const double *cosT; const double *F; double *out;
    int n_rad, N, Lc, lambda_max, ldF, f_off, ld_out, complex_out;
    long long pos_stride;
    double charge; int alt_sign;
    PosMap fmap;
};

// grid: (n_pos, ceil(N*N/256)).  out[p*pos_stride + i*ld_out + j] (real, or complex with zero imaginary part).
__global__ void __launch_bounds__(256) k_direct_assemble(const AsmArgs a) {
    __shared__ double sP[(WP_MAX_LAMBDA + 1) * (2 * WP_MAX_LAMBDA + 1)];
    const int p = blockIdx.x, L = a.lambda_max, ldp = 2 * L + 1;
    if (threadIdx.x == 0) assoc_legendre_all(L, a.cosT[p], sP, ldp);
    __syncthreads();
    const long long idx = ((long long)blockIdx.y * gridDim.z + blockIdx.z) * blockDim.x + threadIdx.x;    // element blocks over (y, z): more than 65 535 of them at N > 4 096
    if (idx >= (long long)a.N * a.N) return;
    const int i = idx / a.N, j = idx % a.N;
    const int ap = a.st_rad[i], lp = a.st_l[i], mp = a.st_m[i];
    const int aa = a.st_rad[j], l = a.st_l[j], m = a.st_m[j];
    const int mu = mp - m, nlm = (a.Lc + 1) * (a.Lc + 1);
    const int alo = min(ap, aa), ahi = max(ap, aa);
    const double *Gp = a.G + ((size_t)lm_index(lp, mp) * nlm + lm_index(l, m)) * (L + 1);
    const double *Fp = a.F + pos_row(a.fmap, p) * a.ldF + a.f_off;
    double acc = 0.0;
    int lam0 = abs(lp - l);
    for (int lam = lam0; lam <= min(lp + l, L); lam += 2) {
        if (abs(mu) > lam) continue;
        int e = a.ent_lookup[((size_t)lam * a.n_rad + alo) * a.n_rad + ahi];
        double term = Gp[lam] * sP[lam * ldp + mu + L] * Fp[e];
        acc += (a.alt_sign && (lam & 1)) ? -term : term;
    }
    const double val = -a.charge * acc;
    const size_t o = (size_t)p * a.pos_stride + (size_t)i * a.ld_out + j;
    if (a.complex_out) { a.out[2 * o] = val; a.out[2 * o + 1] = 0.0; }
    else a.out[o] = val;
}

// Fast path of the assembly: a CTA keeps the pair offsets and the packed state labels in shared memory and loops over
// positions; per position it stages F in pair-major order and the angular factors
//     Ang[lambda][(l'm')][(lm)] = -Z (+-1)^lambda G^lambda_{(l'm'),(lm)} P_lambda^{m'-m}(cos Theta)
// in shared memory, so that every output element is a short dot product of shared-memory operands and the
// global stores are the only HBM traffic (coalesced rows of D).
struct Asm2Args {
    const double *G; const int *pair_off, *ent_perm, *st_pack;
    const double *cosT; const double *F; double *out;
    int n_rad, n_pairs, E, N, Lc, lambda_max, ldF, f_off, ld_out, complex_out, n_pos;
    long long pos_stride;
    double charge; int alt_sign;
    PosMap fmap;
};

// One column j of D over a run of radial functions a_i = a0 .. a1-1 that share l_i (2 l_i + 1 rows each, CNT multipoles
// lambda = lam0, lam0 + 2, .. with this column's l_j), rows mi0 .. mi0 + NMB - 1 of every a_i: the angular factors ang[m_i][k]
// are the same for the whole run and live in registers; per a_i the CNT values F_lambda(a_i, a_j) come from the staged F.
// `ang`, `o` point at row mi0 of the run's first radial function; blockstride = (2 l_i + 1) ostride.
template <int CNT, int NMB, bool CPLX>
__device__ __forceinline__ void asm_run(const double *sF, const int *sOff, const double *ang, int nlm, int nlm2, int a0, int a1, int aj,
                                        int colbase, int n_rad, double *o, size_t ostride, size_t blockstride) {
    double av[NMB][CNT];
    #pragma unroll
    for (int mi = 0; mi < NMB; ++mi)
        #pragma unroll
        for (int k = 0; k < CNT; ++k) av[mi][k] = ang[mi * nlm + k * nlm2];
    int rowbase = a0 * n_rad - a0 * (a0 - 1) / 2 - a0;                            // pair(a_i, a_j) - a_j for a_i <= a_j
    #pragma unroll 1
    for (int ai = a0; ai < a1; ++ai) {
        const double *f = sF + sOff[(ai <= aj) ? rowbase + aj : colbase + ai];
        double fv[CNT];
        #pragma unroll
        for (int k = 0; k < CNT; ++k) fv[k] = f[k];
        double *oo = o;
        #pragma unroll
        for (int mi = 0; mi < NMB; ++mi) {
            double acc = av[mi][0] * fv[0];
            #pragma unroll
            for (int k = 1; k < CNT; ++k) acc = fma(av[mi][k], fv[k], acc);
            if (CPLX) *reinterpret_cast<double2 *>(oo) = make_double2(acc, 0.0); else *oo = acc;
            oo += ostride;
        }
        o += blockstride;
        rowbase += n_rad - ai - 1;
    }
}
// the same for any number of multipoles and rows (angular factors read from shared memory)
template <bool CPLX>
__device__ __forceinline__ void asm_run_any(const double *sF, const int *sOff, const double *ang, int nlm, int nlm2, int cnt, int nmb, int a0, int a1,
                                            int aj, int colbase, int n_rad, double *o, size_t ostride, size_t blockstride) {
    int rowbase = a0 * n_rad - a0 * (a0 - 1) / 2 - a0;
    for (int ai = a0; ai < a1; ++ai) {
        const double *f = sF + sOff[(ai <= aj) ? rowbase + aj : colbase + ai];
        double *oo = o;
        for (int mi = 0; mi < nmb; ++mi) {
            double acc = 0.0;
            for (int k = 0; k < cnt; ++k) acc = fma(ang[mi * nlm + k * nlm2], f[k], acc);
            if (CPLX) *reinterpret_cast<double2 *>(oo) = make_double2(acc, 0.0); else *oo = acc;
            oo += ostride;
        }
        o += blockstride;
        rowbase += n_rad - ai - 1;
    }
}
#define WP_ASM_ARGS sF, sOff, ang, nlm, nlm2, a0, a1, aj, colbase, n_rad, o, ostride, blockstride
template <int NMB, bool CPLX>
__device__ __forceinline__ void asm_run_rows(int cnt, const double *sF, const int *sOff, const double *ang, int nlm, int nlm2, int a0, int a1, int aj,
                                             int colbase, int n_rad, double *o, size_t ostride, size_t blockstride) {
    switch (cnt) {
        case 1: asm_run<1, NMB, CPLX>(WP_ASM_ARGS); break;
        case 2: asm_run<2, NMB, CPLX>(WP_ASM_ARGS); break;
        case 3: asm_run<3, NMB, CPLX>(WP_ASM_ARGS); break;
        case 4: asm_run<4, NMB, CPLX>(WP_ASM_ARGS); break;
        case 5: asm_run<5, NMB, CPLX>(WP_ASM_ARGS); break;
        case 6: asm_run<6, NMB, CPLX>(WP_ASM_ARGS); break;
        default: asm_run_any<CPLX>(sF, sOff, ang, nlm, nlm2, cnt, NMB, a0, a1, aj, colbase, n_rad, o, ostride, blockstride);
    }
}
// all 2 l_i + 1 rows of the run, in blocks of up to four rows
template <bool CPLX>
__device__ __forceinline__ void asm_run_all(int cnt, int nm, const double *sF, const int *sOff, const double *ang, int nlm, int nlm2, int a0, int a1, int aj,
                                            int colbase, int n_rad, double *o, size_t ostride) {
    const size_t blockstride = (size_t)nm * ostride;
    for (int mi0 = 0; mi0 < nm; mi0 += 4) {
        switch (min(4, nm - mi0)) {
            case 1: asm_run_rows<1, CPLX>(cnt, WP_ASM_ARGS); break;
            case 2: asm_run_rows<2, CPLX>(cnt, WP_ASM_ARGS); break;
            case 3: asm_run_rows<3, CPLX>(cnt, WP_ASM_ARGS); break;
            default: asm_run_rows<4, CPLX>(cnt, WP_ASM_ARGS); break;
        }
        ang += 4 * nlm; o += 4 * ostride;
    }
}
#undef WP_ASM_ARGS

constexpr int ASM2_THREADS = 640;          // at most: 102 registers per thread for the register-resident angular factors

template <bool CPLX>
__global__ void __launch_bounds__(ASM2_THREADS) k_direct_assemble2(const Asm2Args a) {
    extern __shared__ __align__(16) double sm2[];
    const int L = a.lambda_max, ldp = 2 * L + 1, nlm = (a.Lc + 1) * (a.Lc + 1), tid = threadIdx.x, nt = blockDim.x;
    double *sF = sm2;                                    // [E] pair-major
    double *sAng = sF + ((a.E + 1) & ~1);                // [L+1][nlm][nlm]
    double *sP = sAng + (size_t)(L + 1) * nlm * nlm;     // [(L+1)][2L+1]
    int *sOff = reinterpret_cast<int *>(sP + (L + 1) * ldp + 1);   // [n_pairs]
    int *sSt = sOff + a.n_pairs;                         // [N]
    int *sRun = sSt + a.N;                               // [n_rad + 1][4]: runs of consecutive radial functions with equal l: a0, a1, l, first row
    __shared__ int s_nrun;
    for (int i = tid; i < a.n_pairs; i += nt) sOff[i] = a.pair_off[i];
    for (int i = tid; i < a.N; i += nt) sSt[i] = a.st_pack[i];
    const int N = a.N, n_rad = a.n_rad;
    __syncthreads();
    if (tid == 0) {
        int nr = 0, i = 0, ai = 0;
        while (ai < n_rad) {
            const int l = (sSt[i] >> 16) & 15, a0 = ai, row0 = i;
            while (ai < n_rad && ((sSt[i] >> 16) & 15) == l) { ++ai; i += 2 * l + 1; if (i >= N) { ai = (i == N) ? ai : n_rad; break; } }
            sRun[4 * nr] = a0; sRun[4 * nr + 1] = ai; sRun[4 * nr + 2] = l; sRun[4 * nr + 3] = row0; ++nr;
            if (i >= N) break;
        }
        s_nrun = nr;
    }
    for (int p = blockIdx.x; p < a.n_pos; p += gridDim.x) {
        __syncthreads();                                 // previous position done with sF / sAng; run table visible
        // P_lambda^mu(cos Theta), one thread per |mu| (independent recurrences in lambda)
        if (tid <= L) {
            const int m = tid;
            const double x = a.cosT[p], sn = sqrt(fmax(0.0, 1.0 - x * x));
            double pmm = 1.0;
            for (int q = 1; q <= m; ++q) pmm = -pmm * (2 * q - 1) * sn;
            double p0 = pmm, p1 = x * (2 * m + 1) * pmm;
            for (int lam = m; lam <= L; ++lam) {
                double val;
                if (lam == m) val = p0;
                else if (lam == m + 1) val = p1;
                else { val = ((2 * lam - 1) * x * p1 - (lam + m - 1) * p0) / (lam - m); p0 = p1; p1 = val; }
                sP[lam * ldp + m + L] = val;
                if (m > 0) {
                    double ratio = 1.0;                      // (lam-m)!/(lam+m)!
                    for (int q = lam - m + 1; q <= lam + m; ++q) ratio /= q;
                    sP[lam * ldp - m + L] = ((m & 1) ? -ratio : ratio) * val;
                }
            }
        }
        const double *Fp = a.F + pos_row(a.fmap, p) * a.ldF + a.f_off;
        #pragma unroll 4
        for (int e = tid; e < a.E; e += nt) sF[a.ent_perm[e]] = Fp[e];
        __syncthreads();
        for (int e = tid; e < (L + 1) * nlm * nlm; e += nt) {
            const int lam = e / (nlm * nlm), r = e - lam * nlm * nlm, lmi = r / nlm, lmj = r - lmi * nlm;
            // (l, m) from the lm index: l = floor(sqrt(lm)), m = lm - l*l - l
            int li = 0; while ((li + 1) * (li + 1) <= lmi) ++li;
            int lj = 0; while ((lj + 1) * (lj + 1) <= lmj) ++lj;
            const int mu = (lmi - li * li - li) - (lmj - lj * lj - lj);
            double v = 0.0;
            if (abs(mu) <= lam) {
                v = a.G[((size_t)lmi * nlm + lmj) * (L + 1) + lam] * sP[lam * ldp + mu + L];
                if (a.alt_sign && (lam & 1)) v = -v;
                v *= -a.charge;
            }
            sAng[e] = v;
        }
        __syncthreads();
        // thread = column j; all threads walk the rows in step, so every store instruction writes one contiguous run of a row of D
        double *outp = a.out + (size_t)p * a.pos_stride * (CPLX ? 2 : 1);
        const int nlm2 = 2 * nlm * nlm, nrun = s_nrun;
        const size_t ostride = (size_t)a.ld_out * (CPLX ? 2 : 1);
        for (int j = tid; j < N; j += nt) {
            const int sj = sSt[j], aj = sj & 0xffff, lj = (sj >> 16) & 15;
            const int colbase = aj * n_rad - aj * (aj - 1) / 2 - aj;              // pair(a_j, a_i) - a_i for a_i >= a_j
            const double *angj = sAng + (sj >> 20);
            double *oj = outp + (size_t)j * (CPLX ? 2 : 1);
            for (int r = 0; r < nrun; ++r) {
                const int a0 = sRun[4 * r], a1 = sRun[4 * r + 1], li = sRun[4 * r + 2], row0 = sRun[4 * r + 3];
                const int lam0 = abs(li - lj), cnt = (min(li + lj, L) - lam0) / 2 + 1;
                const double *ang = angj + (lam0 * nlm + li * li) * nlm;           // lm index of (l_i, -l_i) = l_i^2
                double *o = oj + (size_t)row0 * ostride;
                asm_run_all<CPLX>(cnt, 2 * li + 1, sF, sOff, ang, nlm, nlm2, a0, a1, aj, colbase, n_rad, o, ostride);
            }
        }
    }
}

// ---- a2 alternative: prefix / suffix tables of the grid sum of eq. (7)
// T[g][e] = (P_e[g], Q_e[g]),  P_e[g] = sum_{k=1..g} PP_e[k] r_k^lambda,  Q_e[g] = sum_{k=g+1..Nr} PP_e[k] r_k^-(lambda+1).
struct TabBuildArgs {
    const double *PP[2]; const int *ent_pair[2]; const int *ent_lam; const double *rp, *rm;
    int E[2], E_tot, Nr, Kpad; double2 *T;
};
__global__ void __launch_bounds__(128) k_direct_tables_build(const TabBuildArgs a) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= a.E_tot) return;
    const int c = (e >= a.E[0]) ? 1 : 0, el = e - (c ? a.E[0] : 0), lam = a.ent_lam[e];
    const double *pp = a.PP[c] + (size_t)a.ent_pair[c][el] * a.Kpad;
    const double *rp = a.rp + (size_t)lam * a.Kpad, *rm = a.rm + (size_t)lam * a.Kpad;
    double acc = 0.0;
    a.T[e].x = 0.0;
    for (int k = 1; k <= a.Nr; ++k) { acc += pp[k - 1] * rp[k - 1]; a.T[(size_t)k * a.E_tot + e].x = acc; }
    acc = 0.0;
    a.T[(size_t)a.Nr * a.E_tot + e].y = 0.0;
    for (int k = a.Nr; k >= 1; --k) { acc += pp[k - 1] * rm[k - 1]; a.T[(size_t)(k - 1) * a.E_tot + e].y = acc; }
}

struct TabEvalArgs { const double2 *T; const int *ent_lam; const double *rk, *R; double *F; int E_tot, Nr, ldF, lambda_max, uniform; double h; PosMap rmap, fmap; };
// grid = (positions, entry blocks of 256)
__global__ void __launch_bounds__(256) k_direct_tables_eval(const TabEvalArgs a) {
    __shared__ double sRp[WP_MAX_LAMBDA + 1], sRm[WP_MAX_LAMBDA + 1];
    __shared__ int s_g;
    const int p = blockIdx.x;
    const double R = a.R[pos_row(a.rmap, p)];
    if (threadIdx.x == 0) {
        // g = number of grid points r_k = rk[k-1] (k = 1..Nr) with r_k < R: the same comparison as the GEMM's operand
        int g;
        if (a.uniform) g = (int)floor(R / a.h);
        else { int lo = 0, hi = a.Nr; while (lo < hi) { const int mid = (lo + hi) >> 1; if (a.rk[mid] < R) lo = mid + 1; else hi = mid; } g = lo; }   // bisection on a non-uniform grid
        g = max(0, min(a.Nr, g));
        while (g < a.Nr && a.rk[g] < R) ++g;
        while (g > 0 && !(a.rk[g - 1] < R)) --g;
        s_g = g;
        double Rp = 1.0;
        for (int lam = 0; lam <= a.lambda_max; ++lam) { sRp[lam] = Rp; sRm[lam] = 1.0 / (Rp * R); Rp *= R; }
    }
    __syncthreads();
    const int e = blockIdx.y * blockDim.x + threadIdx.x;
    if (e >= a.E_tot) return;
    const double2 t = a.T[(size_t)s_g * a.E_tot + e];
    const int lam = a.ent_lam[e];
    a.F[pos_row(a.fmap, p) * a.ldF + e] = sRm[lam] * t.x + sRp[lam] * t.y;
}

}  // namespace

extern "C" size_t wpccc_direct_table_bytes(const wpccc_basis *B) {
    return B ? (size_t)(B->Nr + 1) * B->E_tot * sizeof(double2) : 0;
}

extern "C" int wpccc_enable_direct_tables(wpccc_basis *B, void *dev_tables, size_t bytes, void *stream) {
    if (!B) WP_FAIL(WPCCC_EINVAL, "basis is NULL");
    if (!dev_tables) { B->d_dtab = nullptr; return 0; }
    if ((uintptr_t)dev_tables & 255) WP_FAIL(WPCCC_EINVAL, "dev_tables must be 256-byte aligned");
    if (bytes < wpccc_direct_table_bytes(B)) WP_FAIL(WPCCC_ENOMEM, "direct tables need %zu bytes", wpccc_direct_table_bytes(B));
    cudaStream_t s = (cudaStream_t)stream;
    TabBuildArgs a{};
    for (int c = 0; c < B->n_centres; ++c) { a.PP[c] = B->c[c].d_PP; a.ent_pair[c] = B->c[c].d_ent_pair; a.E[c] = B->c[c].E; }
    a.ent_lam = B->d_ent_lam; a.rp = B->d_rp; a.rm = B->d_rm; a.E_tot = B->E_tot; a.Nr = B->Nr; a.Kpad = B->Kpad; a.T = (double2 *)dev_tables;
    k_direct_tables_build<<<(B->E_tot + 127) / 128, 128, 0, s>>>(a);
    WP_CUDA(cudaGetLastError());
    WP_CUDA(cudaStreamSynchronize(s));
    B->d_dtab = (double2 *)dev_tables;
    return 0;
}

int wp_direct_gemm(wpccc_basis *B, int n_pos, const double *d_R, double *d_F, int ldF, cudaStream_t s,
                   const PosMap *rmap, const PosMap *fmap) {
    if (n_pos <= 0) return 0;
    const PosMap ident{0, 0, 0, -1};
    if (B->d_dtab) {
        TabEvalArgs t{};
        t.rmap = rmap ? *rmap : ident; t.fmap = fmap ? *fmap : ident;
        t.T = B->d_dtab; t.ent_lam = B->d_ent_lam; t.rk = B->d_rk; t.R = d_R; t.F = d_F; t.E_tot = B->E_tot; t.Nr = B->Nr; t.ldF = ldF;
        t.lambda_max = B->lambda_max; t.h = B->h; t.uniform = B->d_rgrid == nullptr;
        wp_span_begin(B, FAM_GEMM, s);
        k_direct_tables_eval<<<dim3(n_pos, (B->E_tot + 255) / 256), 256, 0, s>>>(t);
        wp_span_end(B, s, 1);
        WP_CUDA(cudaGetLastError());
        return 0;
    }
    GemmArgs a{};
    a.tiles = B->d_tiles;
    int off = 0;
    for (int c = 0; c < B->n_centres; ++c) {
        a.PP[c] = B->c[c].d_PP; a.ent_pair[c] = B->c[c].d_ent_pair;
        for (int lam = 0; lam <= B->lambda_max + 1; ++lam) a.lam_off[c][lam] = B->c[c].lam_off[lam];
        a.cen_off[c] = off; off += B->c[c].E;
    }
    a.rp = B->d_rp; a.rm = B->d_rm; a.rk = B->d_rk; a.R = d_R; a.F = d_F; a.ldF = ldF; a.n_pos = n_pos; a.Kpad = B->Kpad;
    a.rmap = rmap ? *rmap : ident; a.fmap = fmap ? *fmap : ident;
    const size_t smem = (size_t)NSTG * (BM + BN) * LDS_ * sizeof(double);
    static PerDevice attr_g;
    if (wp_raise(attr_g, smem)) WP_CUDA(cudaFuncSetAttribute(k_direct_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid((n_pos + BM - 1) / BM, (unsigned)B->tiles.size());
    wp_span_begin(B, FAM_GEMM, s);
    k_direct_gemm<<<grid, GEMM_THREADS, smem, s>>>(a);
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}

int wp_direct_assemble(wpccc_basis *B, int c, int n_pos, const double *d_cos, const double *d_F, int ldF,
                       double *d_out, int ld_out, long long pos_stride, int complex_out, cudaStream_t s, const PosMap *fmap) {
    if (n_pos <= 0) return 0;
    const CentreTab &C = B->c[c];
    AsmArgs a{};
    a.fmap = fmap ? *fmap : PosMap{0, 0, 0, -1};
    a.G = C.d_G; a.ent_lookup = C.d_ent_lookup; a.st_rad = C.d_st_rad; a.st_l = C.d_st_l; a.st_m = C.d_st_m;
    a.cosT = d_cos; a.F = d_F; a.out = d_out;
    a.n_rad = C.n_rad; a.N = C.n_states; a.Lc = C.l_max; a.lambda_max = B->lambda_max; a.ldF = ldF;
    a.f_off = (c == 0) ? 0 : B->c[0].E; a.ld_out = ld_out; a.complex_out = complex_out; a.pos_stride = pos_stride;
    // eq. (6): target-centred states see the projectile charge; projectile-centred states see Z_T with (-1)^lambda (A15)
    a.charge = (c == 0) ? B->Z_proj : B->c[0].Z;
    a.alt_sign = (c == 1);
    // fast path when the per-position operands fit shared memory
    const int nlm = (C.l_max + 1) * (C.l_max + 1), L1 = B->lambda_max + 1;
    const size_t smem2 = ((size_t)((C.E + 1) & ~1) + (size_t)L1 * nlm * nlm + (size_t)L1 * (2 * B->lambda_max + 1) + 1) * 8 +
                         ((size_t)C.n_pairs + C.n_states + 4 * ((size_t)C.n_rad + 1)) * 4 + 16;
    if (smem2 <= 220 * 1024) {
        Asm2Args b{};
        b.G = C.d_G; b.pair_off = C.d_pair_off; b.ent_perm = C.d_ent_perm; b.st_pack = C.d_st_pack;
        b.cosT = d_cos; b.F = d_F; b.out = d_out;
        b.n_rad = C.n_rad; b.n_pairs = C.n_pairs; b.E = C.E; b.N = C.n_states; b.Lc = C.l_max; b.lambda_max = B->lambda_max; b.ldF = ldF;
        b.f_off = a.f_off; b.ld_out = ld_out; b.complex_out = complex_out; b.n_pos = n_pos; b.pos_stride = pos_stride;
        b.charge = a.charge; b.alt_sign = a.alt_sign; b.fmap = a.fmap;
        static PerDevice attr2;
        if (wp_raise(attr2, smem2)) {
            WP_CUDA(cudaFuncSetAttribute(k_direct_assemble2<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
            WP_CUDA(cudaFuncSetAttribute(k_direct_assemble2<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
        }
        // one thread per column of D; CTAs of a few positions each, so that the hardware scheduler balances them over whatever
        // SMs the concurrent sweep kernel leaves free
        const int threads = std::min(ASM2_THREADS, (C.n_states + 31) & ~31);
        const int grid = std::max(1, std::min(n_pos, std::max(148 * 8, (n_pos + 3) / 4)));
        wp_span_begin(B, FAM_DASM, s);
        if (complex_out) k_direct_assemble2<true><<<grid, threads, smem2, s>>>(b);
        else k_direct_assemble2<false><<<grid, threads, smem2, s>>>(b);
        wp_span_end(B, s, 1);
        WP_CUDA(cudaGetLastError());
        return 0;
    }
    const long long eb = ((long long)C.n_states * C.n_states + 255) / 256;
    const unsigned gz = (unsigned)((eb + 65534) / 65535);
    dim3 grid(n_pos, (unsigned)((eb + gz - 1) / gz), gz);
    wp_span_begin(B, FAM_DASM, s);
    k_direct_assemble<<<grid, 256, 0, s>>>(a);
    wp_span_end(B, s, 1);
    WP_CUDA(cudaGetLastError());
    return 0;
}
