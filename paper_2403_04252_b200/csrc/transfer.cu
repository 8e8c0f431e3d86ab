// Two-centre overlap and electron-transfer elements: eq. (8)-(9) structure of the paper in the
// body-frame cylindrical Gauss-Legendre form fixed by BASELINE.json configs[1], [3] (A1, A4, A5, A10).
//
// Per projectile position (b, z, v), with R = |R|, Theta = angle(R, v):
//   body-frame integrals over the (rho', z') product nodes with the discrete azimuthal sum Phi_Delta folded in
//     Sb [(b,q'),(a,q)] = sum_{i,k} W_ik e^{-i v cosTh (z'_k - R/2)} Phi_{q-q'}(v sinTh rho'_i) B_{bq'}(i,k) A_{aq}(i,k)
//     Hb [(b,q'),(a,q)] = same with A -> Ah = -(Z_P/r_P) A + Ag                       (H_PT)
//     Tb [(b,q'),(a,q)] = same with B -> Bh = -(Z_T/r_T) B + Bg;  H_TP^body = conj(Tb)^T
//   A_{aq} = u_a(r_T)/r_T Theta~_{l_a q}(cos th'_T),  B_{bq'} = u_b(r_P)/r_P Theta~_{l_b q'}(cos th'_P),
//   radial functions by five-point Lagrange interpolation on the r-grid.
//   Then the Wigner rotation of eq. (8):  X_lab = d(Theta) X_body d(Theta)^T per (l_b, l_a) block.
//
// What this file does differently from a literal evaluation:
//   * the weight separates, W Phi e^{..} = [w_rho rho Phi_Delta(i)] [w_z e^{..}(k)]: the z'-sum is one uniform
//     complex-weighted GEMM per ring i (FP64 DMMA), the Delta-dependent ring weight is applied to its result;
//   * Theta~_{l,-q} = (-1)^q Theta~_{lq} and Phi_{-Delta} = Phi_Delta (the phi' nodes are symmetric about pi), so
//     only q, q' >= 0 columns are tabulated and contracted; the two families Phi_{|q-q'|} and Phi_{q+q'} of ring
//     weights rebuild all sign combinations;
//   * Phi^+_{-Delta} = conj(Phi^-_Delta) and the axial phases are conjugate, so H_TP shares the weights of S_PT.
#include "common.cuh"
#include "ptx.cuh"

namespace {

constexpr int MAXD = 2 * WP_MAX_L;          // largest Delta
constexpr int NLQ = (WP_MAX_L + 1) * (WP_MAX_L + 2) / 2;
__host__ __device__ inline int lq_index(int l, int q) { return l * (l + 1) / 2 + q; }

__constant__ double c_fact[2 * WP_MAX_L + 2];
__constant__ double c_thnorm[NLQ];          // sqrt((2l+1)/2 (l-q)!/(l+q)!)

// Evaluated positions of a launch group (TransferSel in common.cuh): compact index q -> window position p.
struct SelDev { int n_c, n_idx, n_pre, suf0; };          // n_idx == 0: identity
__device__ __forceinline__ int sel_pos(const SelDev &s, int q) {
    if (s.n_idx == 0) return q;
    const int g = q / s.n_c, lj = q - g * s.n_c;
    return g * s.n_idx + (lj < s.n_pre ? lj : lj - s.n_pre + s.suf0);
}

// ------------------------------------------------------------------------------------------------ per-position tables
struct PosTabs {      // layout of the small per-position table block (doubles), filled by k_tpos
    int n_rho, n_z, n_phi, dmax;
    __host__ __device__ int off_zq() const { return 0; }                       // z'_k                 [n_z]
    __host__ __device__ int off_ck() const { return n_z; }                     // w_z e^{-i v cosTh (z'-R/2)}  [n_z][2]
    __host__ __device__ int off_rho() const { return 3 * n_z; }                // rho'_i               [n_rho]
    __host__ __device__ int off_rw() const { return 3 * n_z + n_rho; }         // w_rho rho Phi_d(i)   [dmax+1][n_rho][2]
    __host__ __device__ int size() const { return (3 * n_z + n_rho + 2 * (dmax + 1) * n_rho + 3) & ~3; }
};

struct TposArgs {
    PosTabs L; const double *R, *cosT, *sinT, *v; const double *gl_rho, *gl_phi, *gl_zq, *gl_zh;
    double rho_max, z_pad; int phi_rule; double *out;
    SelDev sel; int q0;                      // block x evaluates window position sel_pos(sel, q0 + x)
};

// grid = positions, block = 128
__global__ void __launch_bounds__(128) k_tpos(const TposArgs a) {
    const int p = blockIdx.x, tid = threadIdx.x, gp = sel_pos(a.sel, a.q0 + p);
    const PosTabs &L = a.L;
    double *o = a.out + (size_t)p * L.size();
    const double R = a.R[gp], cT = a.cosT[gp], sT = a.sinT[gp], v = a.v[gp];
    const int nq = L.n_z / 4, nh = L.n_z / 2;
    for (int k = tid; k < L.n_z; k += blockDim.x) {
        double lo, hi, x, w;
        if (k < nq) { lo = -a.z_pad; hi = 0.0; x = a.gl_zq[k]; w = a.gl_zq[nq + k]; }
        else if (k < nq + nh) { lo = 0.0; hi = R; x = a.gl_zh[k - nq]; w = a.gl_zh[nh + k - nq]; }
        else { lo = R; hi = __dadd_rn(R, a.z_pad); x = a.gl_zq[k - nq - nh]; w = a.gl_zq[nq + k - nq - nh]; }
        const double half = __dmul_rn(0.5, __dsub_rn(hi, lo)), mid = __dmul_rn(0.5, __dadd_rn(hi, lo));
        const double zk = __dadd_rn(__dmul_rn(half, x), mid), wz = __dmul_rn(half, w);
        double sn, cs; sincos(-(v * cT) * (zk - 0.5 * R), &sn, &cs);
        o[L.off_zq() + k] = zk;
        o[L.off_ck() + 2 * k] = wz * cs; o[L.off_ck() + 2 * k + 1] = wz * sn;
    }
    const double twopi = 6.283185307179586476925286766559;
    for (int i = tid; i < L.n_rho; i += blockDim.x) {
        const double half = __dmul_rn(0.5, a.rho_max);
        const double rho = __dadd_rn(__dmul_rn(half, a.gl_rho[i]), half), wr = __dmul_rn(__dmul_rn(half, a.gl_rho[L.n_rho + i]), rho);
        o[L.off_rho() + i] = rho;
        const double x = (v * sT) * rho;
        double sr[MAXD + 1], si[MAXD + 1];
        for (int d = 0; d <= L.dmax; ++d) { sr[d] = 0.0; si[d] = 0.0; }
        const int nphi = a.phi_rule ? 512 : L.n_phi;
        for (int j = 0; j < nphi; ++j) {
            double phi, wj;
            if (a.phi_rule) { phi = twopi * (double)j / 512.0; wj = twopi / 512.0; }
            else { phi = __dadd_rn(__dmul_rn(0.5 * twopi, a.gl_phi[j]), 0.5 * twopi); wj = __dmul_rn(0.5 * twopi, a.gl_phi[L.n_phi + j]); }
            double s1, c1; sincos(phi, &s1, &c1);
            double sx, cx; sincos(x * c1, &sx, &cx);          // e^{+i x cos phi}
            for (int d = 0; d <= L.dmax; ++d) {
                double sd, cd; sincos((double)d * phi, &sd, &cd);
                sr[d] += wj * (cd * cx - sd * sx); si[d] += wj * (cd * sx + sd * cx);
            }
        }
        for (int d = 0; d <= L.dmax; ++d) {
            o[L.off_rw() + 2 * (d * L.n_rho + i)] = wr * sr[d] / twopi;
            o[L.off_rw() + 2 * (d * L.n_rho + i) + 1] = wr * si[d] / twopi;
        }
    }
}

// ------------------------------------------------------------------------------------------------ node tables (a4)
// Table of one side for one position, fragment-major for m8n8k4:  T[tile][ring][kc][c8][32] with
//   column = tile*64 + c8*8 + lane/4,  z' node k = kc*4 + lane%4.
// Columns: [X (nqc, padded to nq8) | Xh (nq8)], X = A (side 0, centre T) or B (side 1, centre P).
// Padding columns are never written: the caller zeroes the table buffer once.
struct TtabArgs {
    PosTabs L; const double *pos;            // per-position tables
    const double *R;
    const double *Ut[2]; const int *lrad[2]; int n_rad[2], nf_pad[2], nq8[2], ntile[2];
    const int *colidx[2];                    // [n_rad][WP_MAX_L+1] column of (a, q) or -1
    double Zother[2];                        // side 0 (T functions): Z_P;  side 1: Z_T
    double h; int Nr, KC;                    // KC: z' nodes per CTA (multiple of 4)
    int sph;                                 // 1: spheroidal nodes: ring = eta_i (pos[off_rho]), axial node = tau_k (pos[off_zq])
    const double *rgrid;                     // [Nr+1] non-uniform radial grid, or nullptr (uniform r_k = k h)
    double *out[2]; size_t pos_stride[2];    // doubles per position for each side
    int lmax[2];
    SelDev sel; int q0;
};

__device__ __forceinline__ void st_global_256(double *p, const double (&v)[4]) {       // p 32-byte aligned (sm_100: STG.256)
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};\n" ::"l"(p), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[3]) : "memory");
}

// grid = (ring * n_kchunks, side, position), block = 256, dynamic smem (per-node quantities only).
// Phase 1: one thread per node: geometry, Lagrange weights, Theta~_{lq}.  Phase 2: a warp takes a k4-group of 4 nodes,
// lane = radial function: it interpolates (u_a, g_a) at the four nodes with one 16-byte load per stencil point and
// stores X, Xh for q = 0..l_a straight into the fragment-major table, 32 bytes (4 nodes of one column) per store.
__global__ void __launch_bounds__(256) k_ttab(const TtabArgs a) {
    extern __shared__ __align__(16) double sm[];
    const int side = blockIdx.y, p = blockIdx.z, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nkch = a.L.n_z / a.KC, ring = blockIdx.x / nkch, k0 = (blockIdx.x % nkch) * a.KC, KC = a.KC;
    const int nq8 = a.nq8[side], lmax = a.lmax[side];
    const int nlq = (lmax + 1) * (lmax + 2) / 2;
    double *sLag = sm;                                   // [5][KC]
    double *sRinv = sLag + 5 * KC, *sPot = sRinv + KC;   // [KC] 1/r_side, -Z_other/r_other
    double *sTh = sPot + KC;                             // [nlq][KC]
    int *sJ = reinterpret_cast<int *>(sTh + (size_t)nlq * KC);   // [KC] stencil centre, -1 beyond r_max
    const double *pt = a.pos + (size_t)p * a.L.size();
    const double R = a.R[sel_pos(a.sel, a.q0 + p)];
    const int nkc = a.L.n_z / 4;
    const int tile_stride = a.L.n_rho * nkc * 256;

    if (tid < KC) {
        const double rho = pt[a.L.off_rho() + ring], zk = pt[a.L.off_zq() + k0 + tid];
        double rs, ro, c;
        if (a.sph) {
            // eq. (9): r_T = R (eta + tau)/2, r_P = R (eta - tau)/2, cos th'_T = (eta tau + 1)/(eta + tau), cos th'_P = (eta tau - 1)/(eta - tau)
            const double eta = rho, tau = zk, hR = __dmul_rn(0.5, R), et = __dmul_rn(eta, tau);
            const double sp = __dadd_rn(eta, tau), sm_ = __dsub_rn(eta, tau);
            const double rT = __dmul_rn(hR, sp), rP = __dmul_rn(hR, sm_);
            rs = side ? rP : rT; ro = side ? rT : rP;
            c = side ? __dsub_rn(et, 1.0) / sm_ : __dadd_rn(et, 1.0) / sp;
        } else {
            const double zP = __dsub_rn(zk, R);
            const double rT = sqrt(__dadd_rn(__dmul_rn(rho, rho), __dmul_rn(zk, zk)));
            const double rP = sqrt(__dadd_rn(__dmul_rn(rho, rho), __dmul_rn(zP, zP)));
            rs = side ? rP : rT; ro = side ? rT : rP;
            c = (side ? zP : zk) / rs;
        }
        int j;
        if (a.rgrid) {
            // non-uniform grid ("denser around the origin"): stencil centre = the nearest grid point (the lower one on a
            // tie), by bisection; five-point Lagrange weights on the actual abscissae
            int lo = 0, hi = a.Nr;                               // invariant: r[lo] <= rs (or lo == 0), r[hi] > rs (or hi == Nr)
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (a.rgrid[mid] <= rs) lo = mid; else hi = mid; }
            j = (__dsub_rn(rs, a.rgrid[lo]) <= __dsub_rn(a.rgrid[hi], rs)) ? lo : hi;
            j = max(2, min(a.Nr - 2, j));
            double x[5];
            #pragma unroll
            for (int q = 0; q < 5; ++q) x[q] = a.rgrid[j - 2 + q];
            #pragma unroll
            for (int q = 0; q < 5; ++q) {
                double L = 1.0;
                #pragma unroll
                for (int c = 0; c < 5; ++c) if (c != q) L = L * (rs - x[c]) / (x[q] - x[c]);
                sLag[q * KC + tid] = L;
            }
            sJ[tid] = (rs > a.rgrid[a.Nr]) ? -1 : j;
        } else {
            j = (int)floor(rs / a.h + 0.5);
            j = max(2, min(a.Nr - 2, j));
            const double t = rs / a.h - (double)j;
            // Lagrange basis on offsets -2..2
            sLag[0 * KC + tid] = (t + 1.0) * t * (t - 1.0) * (t - 2.0) / 24.0;
            sLag[1 * KC + tid] = -(t + 2.0) * t * (t - 1.0) * (t - 2.0) / 6.0;
            sLag[2 * KC + tid] = (t + 2.0) * (t + 1.0) * (t - 1.0) * (t - 2.0) / 4.0;
            sLag[3 * KC + tid] = -(t + 2.0) * (t + 1.0) * t * (t - 2.0) / 6.0;
            sLag[4 * KC + tid] = (t + 2.0) * (t + 1.0) * t * (t - 1.0) / 24.0;
            sJ[tid] = (rs > a.Nr * a.h) ? -1 : j;
        }
        sRinv[tid] = 1.0 / rs;
        sPot[tid] = -a.Zother[side] / ro;
        // Theta~_{lq}(c), q >= 0
        const double s = sqrt(fmax(0.0, __dsub_rn(1.0, __dmul_rn(c, c))));
        double pmm = 1.0;
        for (int q = 0; q <= lmax; ++q) {
            if (q > 0) pmm = -pmm * (2 * q - 1) * s;
            double p0 = pmm, p1 = c * (2 * q + 1) * pmm;
            for (int l = q; l <= lmax; ++l) {
                double val;
                if (l == q) val = p0;
                else if (l == q + 1) val = p1;
                else { val = ((2 * l - 1) * c * p1 - (l + q - 1) * p0) / (l - q); p0 = p1; p1 = val; }
                sTh[lq_index(l, q) * KC + tid] = c_thnorm[lq_index(l, q)] * val;
            }
        }
    }
    __syncthreads();
    const double2 *Ut = reinterpret_cast<const double2 *>(a.Ut[side]);
    const int nr = a.n_rad[side], nf2 = a.nf_pad[side] / 2;        // row stride in (u, g) pairs
    double *out = a.out[side] + (size_t)p * a.pos_stride[side];
    // lane = radial function: a stencil row of all functions is ONE contiguous run per request (16 n_rad bytes), and a
    // lane owns the four z' nodes of its columns in a k4-group, i.e. one whole 32-byte sector per (column, k4-group),
    // written with a single 256-bit store
    for (int kcl = warp; kcl < KC / 4; kcl += 8) {
        double *dst = out + ((size_t)ring * nkc + (k0 / 4 + kcl)) * 256;
        for (int aa = lane; aa < nr; aa += 32) {
            double fu[4], fg[4], pt4[4];
            #pragma unroll
            for (int kn = 0; kn < 4; ++kn) {
                const int n = kcl * 4 + kn, j = sJ[n];
                fu[kn] = 0.0; fg[kn] = 0.0; pt4[kn] = sPot[n];
                if (j >= 0) {
                    const double L0 = sLag[n], L1 = sLag[KC + n], L2 = sLag[2 * KC + n], L3 = sLag[3 * KC + n], L4 = sLag[4 * KC + n];
                    const double rinv = sRinv[n];
                    const double2 *row = Ut + (size_t)(j - 2) * nf2 + aa;
                    const double2 v0 = row[0], v1 = row[nf2], v2 = row[2 * nf2], v3 = row[3 * nf2], v4 = row[4 * nf2];
                    double u = L0 * v0.x, g = L0 * v0.y;
                    u += L1 * v1.x; g += L1 * v1.y;
                    u += L2 * v2.x; g += L2 * v2.y;
                    u += L3 * v3.x; g += L3 * v3.y;
                    u += L4 * v4.x; g += L4 * v4.y;
                    fu[kn] = u * rinv; fg[kn] = g * rinv;
                }
            }
            const int l = a.lrad[side][aa];
            const int *cix = a.colidx[side] + aa * (WP_MAX_L + 1);
            const double *th_l = sTh + (size_t)lq_index(l, 0) * KC + kcl * 4;
            for (int q = 0; q <= l; ++q) {
                const int col = cix[q], colh = nq8 + col;
                double X[4], Xh[4];
                #pragma unroll
                for (int kn = 0; kn < 4; ++kn) {
                    const double th = th_l[q * KC + kn];
                    const double Xg = fg[kn] * th;
                    X[kn] = fu[kn] * th; Xh[kn] = pt4[kn] * X[kn] + Xg;
                }
                st_global_256(dst + (size_t)(col >> 6) * tile_stride + (col & 63) * 4, X);
                st_global_256(dst + (size_t)(colh >> 6) * tile_stride + (colh & 63) * 4, Xh);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ contraction (a5)
// TMA ring of the contraction: 3 stages of 16 k4-groups of z' nodes per operand (256 doubles each), 192 KB.
// Mirror-pair kernel (DUAL): the 64 accumulators per thread of the mirror position (128 KB per CTA; the register file
// holds the 96 of the position itself) live in tensor memory, 256 of the SM's 512 TMEM columns, moved with
// tcgen05.ld / tcgen05.st in the per-ring epilogue: neither registers nor shared-memory bandwidth are spent on them.
template <bool DUAL> struct TcRing {
    static constexpr int STAGES = 3, KCS = 16, STAGE_DOUBLES = KCS * 256;
    static constexpr size_t ACC_DOUBLES = 0;
    static constexpr int TMEM_COLS = 256;
};

// 16 consecutive 32-bit TMEM columns of this thread's lane (shape 32x32b: lane = 32 (warp % 4) + laneid) <-> 8 doubles
__device__ __forceinline__ void tmem_ld8(unsigned taddr, double (&d)[8]) {
    unsigned r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
    #pragma unroll
    for (int k = 0; k < 8; ++k) d[k] = __hiloint2double((int)r[2 * k + 1], (int)r[2 * k]);
}
__device__ __forceinline__ void tmem_st8(unsigned taddr, const double (&d)[8]) {
    unsigned r[16];
    #pragma unroll
    for (int k = 0; k < 8; ++k) { r[2 * k] = (unsigned)__double2loint(d[k]); r[2 * k + 1] = (unsigned)__double2hiint(d[k]); }
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};\n"
                 :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
                    "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }

struct TconArgs {
    PosTabs L; const double *pos;
    const double *tabT, *tabP; size_t strideT, strideP;         // node tables (doubles per position)
    int nq8T, nq8P, ntT, ntP;                                    // padded half widths, number of 64-tiles
    const int *qT, *qP;                                          // [nq8] q of column (q >= 0), -1 padding
    const int2 *tiles; int n_tiles;                              // (row tile over [B|Bh], col tile over [A|Ah])
    int n_split;                                                 // ring splits
    double *part;                                                // [p][split][fam 2][prod 3][nq8P][nq8T] complex
    // DUAL: block z = compact position q0 + z; its mirror's integrals go to the stash slot (n_split == 1)
    SelDev sel; int q0, n_st; long long i0, i_mid; double *stash;
};

// One stage (nk k4-groups of z' nodes) of a warp's 16 x 8 NJ complex tile: C += (B ck)^T A with the complex weight
// ck = w_z e^{..} folded into the B fragments.  ALL: every 8 x 8 sub-tile is needed (no predicates in the loop);
// FULL: nk == TC_KCS (fully unrolled, fragments of the next k4-group loaded while the current DMMAs issue).
template <int NJ, bool ALL, bool FULL, int TC_KCS>
__device__ __forceinline__ void tcon_stage(const double *Ab, const double *Bb, const double *ck, int nk, const bool (&need)[2][NJ],
                                           double (&Cre)[2][NJ][2], double (&Cim)[2][NJ][2]) {
    double af[2][NJ], bb[2][2], cc[2][2];
    auto load = [&](int s, int kc) {
        #pragma unroll
        for (int j = 0; j < NJ; ++j) af[s][j] = Ab[kc * 256 + j * 32];
        #pragma unroll
        for (int i = 0; i < 2; ++i) bb[s][i] = Bb[kc * 256 + i * 32];
        cc[s][0] = ck[8 * kc]; cc[s][1] = ck[8 * kc + 1];
    };
    auto mma = [&](int s) {
        double br[2], bi[2];
        #pragma unroll
        for (int i = 0; i < 2; ++i) { br[i] = bb[s][i] * cc[s][0]; bi[i] = bb[s][i] * cc[s][1]; }
        #pragma unroll
        for (int i = 0; i < 2; ++i)
            #pragma unroll
            for (int j = 0; j < NJ; ++j)
                if (ALL || need[i][j]) {
                    dmma884(Cre[i][j][0], Cre[i][j][1], br[i], af[s][j]);
                    dmma884(Cim[i][j][0], Cim[i][j][1], bi[i], af[s][j]);
                }
    };
    if (FULL) {
        load(0, 0);
        #pragma unroll
        for (int kc = 0; kc < TC_KCS; ++kc) {
            if (kc + 1 < TC_KCS) load((kc + 1) & 1, kc + 1);
            mma(kc & 1);
        }
    } else {
        #pragma unroll 2
        for (int kc = 0; kc < nk; ++kc) { load(0, kc); mma(0); }
    }
}

// grid = (tile, ring split, position); block = 4 (rows) x 8/NJ (cols) warps; warp tile 16 x 8 NJ complex
// (NJ = 4: 8 warps, NJ = 2: 16 warps).  Stages are released per warp through `empty` mbarriers (no block-wide
// barrier in the main loop); thread 0 refills the buffer of stage st - 1 once it has finished stage st itself.
template <int NJ, bool DUAL>
__global__ void __launch_bounds__(128 * (8 / NJ), 1) k_tcon(const TconArgs a) {
    constexpr int WC = 8 / NJ, NW = 4 * WC, TC_THREADS = 32 * NW;
    constexpr int TC_STAGES = TcRing<DUAL>::STAGES, TC_KCS = TcRing<DUAL>::KCS, TC_STAGE_DOUBLES = TcRing<DUAL>::STAGE_DOUBLES;
    static_assert(!DUAL || NJ == 4, "mirror-pair kernel: 256 threads");
    extern __shared__ __align__(128) double sm[];
    double *sA = sm;                                          // [STAGES][TC_STAGE_DOUBLES]  A-side (mma "B" operand)
    double *sB = sA + TC_STAGES * TC_STAGE_DOUBLES;           // [STAGES][TC_STAGE_DOUBLES]  B-side (mma "A" operand)
    __shared__ unsigned s_tmem;                               // DUAL: base address of the allocated TMEM columns
    double *sCk = sB + TC_STAGES * TC_STAGE_DOUBLES + TcRing<DUAL>::ACC_DOUBLES;      // [n_z][2]
    double *sRw = sCk + 2 * a.L.n_z;                          // [dmax+2][n_rho][2], last row zero (weight of unused elements)
    __shared__ __align__(8) unsigned long long bar[TC_STAGES], empty[TC_STAGES];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int p = blockIdx.z, split = blockIdx.y;
    const int2 tl = a.tiles[blockIdx.x];
    const int rt = tl.x, ct = tl.y;
    const double *pt = a.pos + (size_t)p * a.L.size();
    const int n_rho = a.L.n_rho, n_z = a.L.n_z, nkc = n_z / 4;
    const int ring0 = (int)((long long)n_rho * split / a.n_split), ring1 = (int)((long long)n_rho * (split + 1) / a.n_split);
    const int spr = (nkc + TC_KCS - 1) / TC_KCS;              // stages per ring
    const int n_st = (ring1 - ring0) * spr;

    for (int i = tid; i < 2 * n_z; i += TC_THREADS) sCk[i] = pt[a.L.off_ck() + i];
    for (int i = tid; i < 2 * (a.L.dmax + 1) * n_rho; i += TC_THREADS) sRw[i] = pt[a.L.off_rw() + i];
    for (int i = tid; i < 2 * n_rho; i += TC_THREADS) sRw[2 * (a.L.dmax + 1) * n_rho + i] = 0.0;
    if (DUAL && tid < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&s_tmem)), "n"(TcRing<DUAL>::TMEM_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::);
    }
    if (tid == 0) { for (int s = 0; s < TC_STAGES; ++s) { mbar_init(&bar[s], 1); mbar_init(&empty[s], NW); } asm volatile("fence.mbarrier_init.release.cluster;\n" ::); }
    if (DUAL) asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    unsigned tacc = 0;            // DUAL: this thread's 128 TMEM columns: lane 32 (warp % 4) + laneid, columns 128 (warp / 4) ..
    if (DUAL) {
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
        tacc = s_tmem + ((unsigned)(32 * (warp & 3)) << 16) + (unsigned)(128 * (warp >> 2));
        const double zero[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        #pragma unroll
        for (int k = 0; k < 2 * NJ; ++k) tmem_st8(tacc + 16 * k, zero);
        tmem_wait_st();
    }

    const double *gA = a.tabT + (size_t)p * a.strideT + (size_t)ct * n_rho * nkc * 256;
    const double *gB = a.tabP + (size_t)p * a.strideP + (size_t)rt * n_rho * nkc * 256;
    auto issue = [&](int st) {
        const int ring = ring0 + st / spr, kc0 = (st % spr) * TC_KCS, nk = min(TC_KCS, nkc - kc0), buf = st % TC_STAGES;
        const unsigned bytes = (unsigned)nk * 256 * 8;
        mbar_expect_tx(&bar[buf], 2 * bytes);
        tma_bulk_g2s(sA + buf * TC_STAGE_DOUBLES, gA + ((size_t)ring * nkc + kc0) * 256, bytes, &bar[buf]);
        tma_bulk_g2s(sB + buf * TC_STAGE_DOUBLES, gB + ((size_t)ring * nkc + kc0) * 256, bytes, &bar[buf]);
    };
    if (tid == 0) for (int st = 0; st < min(TC_STAGES, n_st); ++st) issue(st);

    const int wr = warp / WC, wc = warp % WC;                 // warp rows 16*wr.., cols 8*NJ*wc..
    const int fr = lane >> 2, fk = lane & 3;
    // per-thread output bookkeeping: element (i, j, e): row = rt*64 + 16 wr + 8 i + fr, col = ct*64 + 8 NJ wc + 8 j + 2 fk + e
    // needed sub-tiles: not (Bh x Ah)
    bool need[2][NJ];
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int r8 = rt * 64 + 16 * wr + 8 * i, c8 = ct * 64 + 8 * NJ * wc + 8 * j;
            need[i][j] = (r8 < 2 * a.nq8P) && (c8 < 2 * a.nq8T) && !(r8 >= a.nq8P && c8 >= a.nq8T);
        }
    bool any_need = false, all_need = true;
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < NJ; ++j) { any_need |= need[i][j]; all_need &= need[i][j]; }

    double Cre[2][NJ][2], Cim[2][NJ][2], Mre[2][NJ][2], Mim[2][NJ][2], Pre[2][NJ][2], Pim[2][NJ][2];
    int dm[2][NJ][2], dp[2][NJ][2];                          // offsets of the ring-weight rows in sRw (zero row if unused)
    unsigned okmask = 0;                                     // bit (i NJ + j) 2 + e: element is a wanted output
    const int zrow = 2 * (a.L.dmax + 1) * n_rho;
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < NJ; ++j)
            #pragma unroll
            for (int e = 0; e < 2; ++e) {
                Cre[i][j][e] = Cim[i][j][e] = Mre[i][j][e] = Mim[i][j][e] = Pre[i][j][e] = Pim[i][j][e] = 0.0;
                const int gr = rt * 64 + 16 * wr + 8 * i + fr, gc = ct * 64 + 8 * NJ * wc + 8 * j + 2 * fk + e;
                int qp = -1, qq = -1;
                if (gr < 2 * a.nq8P) qp = a.qP[gr % a.nq8P];
                if (gc < 2 * a.nq8T) qq = a.qT[gc % a.nq8T];
                const bool ok = need[i][j] && qp >= 0 && qq >= 0;
                if (ok) okmask |= 1u << ((i * NJ + j) * 2 + e);
                dm[i][j][e] = ok ? 2 * abs(qq - qp) * n_rho : zrow;
                dp[i][j][e] = (ok && qp > 0 && qq > 0) ? 2 * (qq + qp) * n_rho : zrow;
            }

    for (int st = 0; st < n_st; ++st) {
        const int buf = st % TC_STAGES, ring = ring0 + st / spr, kc0 = (st % spr) * TC_KCS, nk = min(TC_KCS, nkc - kc0);
        mbar_wait(&bar[buf], (st / TC_STAGES) & 1);
        if (any_need) {
            const double *Ab = sA + buf * TC_STAGE_DOUBLES + (NJ * wc) * 32 + lane;
            const double *Bb = sB + buf * TC_STAGE_DOUBLES + (2 * wr) * 32 + lane;
            const double *ck = sCk + 2 * (kc0 * 4 + fk);
            if (all_need && nk == TC_KCS) tcon_stage<NJ, true, true, TC_KCS>(Ab, Bb, ck, nk, need, Cre, Cim);
            else if (all_need) tcon_stage<NJ, true, false, TC_KCS>(Ab, Bb, ck, nk, need, Cre, Cim);
            else if (nk == TC_KCS) tcon_stage<NJ, false, true, TC_KCS>(Ab, Bb, ck, nk, need, Cre, Cim);      // ragged tile: same unrolled pipeline, warp-uniform predicates
            else tcon_stage<NJ, false, false, TC_KCS>(Ab, Bb, ck, nk, need, Cre, Cim);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[buf]);           // this warp is done with the buffer
        if (tid == 0 && st >= 1 && st - 1 + TC_STAGES < n_st) {
            mbar_wait(&empty[(st - 1) % TC_STAGES], ((st - 1) / TC_STAGES) & 1);
            issue(st - 1 + TC_STAGES);
        }
        if ((st % spr) == spr - 1) {
            // ring epilogue (branch-free): acc(-) += w_rho rho Phi_{|q-q'|}(ring) C,  acc(+) += w_rho rho Phi_{q+q'}(ring) C
            const double2 *rw = reinterpret_cast<const double2 *>(sRw) + ring;
            #pragma unroll
            for (int i = 0; i < 2; ++i)
                #pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    double mir[8];       // DUAL, per e: B of family (-) and of family (+), see below
                    if (DUAL) tmem_ld8(tacc + 16 * (i * NJ + j), mir);
                    #pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const double cr = Cre[i][j][e], ci = Cim[i][j][e];
                        const double2 wm = rw[dm[i][j][e] >> 1], wp = rw[dp[i][j][e] >> 1];
                        if (DUAL) {
                            // The mirror position has the same ring weight and the conjugate z'-sum, w (cr - i ci).  With
                            // A = sum_ring w cr (registers) and B = sum_ring w ci (tensor memory), both complex, the pair is
                            // M = A + i B and M' = A - i B: eight plain fma per element and ring for both positions.
                            Mre[i][j][e] = fma(wm.x, cr, Mre[i][j][e]); Mim[i][j][e] = fma(wm.y, cr, Mim[i][j][e]);
                            Pre[i][j][e] = fma(wp.x, cr, Pre[i][j][e]); Pim[i][j][e] = fma(wp.y, cr, Pim[i][j][e]);
                            mir[4 * e + 0] = fma(wm.x, ci, mir[4 * e + 0]); mir[4 * e + 1] = fma(wm.y, ci, mir[4 * e + 1]);
                            mir[4 * e + 2] = fma(wp.x, ci, mir[4 * e + 2]); mir[4 * e + 3] = fma(wp.y, ci, mir[4 * e + 3]);
                        } else {
                            Mre[i][j][e] += wm.x * cr - wm.y * ci; Mim[i][j][e] += wm.x * ci + wm.y * cr;
                            Pre[i][j][e] += wp.x * cr - wp.y * ci; Pim[i][j][e] += wp.x * ci + wp.y * cr;
                        }
                        Cre[i][j][e] = 0.0; Cim[i][j][e] = 0.0;
                    }
                    if (DUAL) tmem_st8(tacc + 16 * (i * NJ + j), mir);
                }
            if (DUAL) tmem_wait_st();
        }
    }
    // write partial sums
    const size_t blk = (size_t)a.nq8P * a.nq8T;
    double *o = a.part + ((size_t)p * a.n_split + split) * 6 * blk * 2;
    double *om = nullptr;                                   // stash slot of the mirror position
    if (DUAL && a.stash) {
        const int q = a.q0 + p, g = a.sel.n_idx ? q / a.sel.n_c : 0;
        const long long i = a.i0 + (sel_pos(a.sel, q) - g * a.sel.n_idx);
        if (i < a.i_mid && i >= a.i_mid - a.n_st) om = a.stash + ((size_t)g * a.n_st + (size_t)(a.i_mid - i - 1)) * 6 * blk * 2;
    }
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < NJ; ++j) {
            double mir[8];
            if (DUAL) tmem_ld8(tacc + 16 * (i * NJ + j), mir);       // warp-uniform: outside the per-element predicate
            #pragma unroll
            for (int e = 0; e < 2; ++e) {
                if (!((okmask >> ((i * NJ + j) * 2 + e)) & 1u)) continue;
                const int gr = rt * 64 + 16 * wr + 8 * i + fr, gc = ct * 64 + 8 * NJ * wc + 8 * j + 2 * fk + e;
                const int hr = gr / a.nq8P, ir = gr % a.nq8P, hc = gc / a.nq8T, ic = gc % a.nq8T;
                const int prod = hr ? 2 : (hc ? 1 : 0);
                const size_t idx = ((size_t)prod * blk + (size_t)ir * a.nq8T + ic) * 2;
                double *op = o + 3 * blk * 2;
                if (DUAL) {          // M = A + i B here, M' = A - i B for the mirror position
                    o[idx] = Mre[i][j][e] - mir[4 * e + 1]; o[idx + 1] = Mim[i][j][e] + mir[4 * e];
                    op[idx] = Pre[i][j][e] - mir[4 * e + 3]; op[idx + 1] = Pim[i][j][e] + mir[4 * e + 2];
                    if (om) {
                        om[idx] = Mre[i][j][e] + mir[4 * e + 1]; om[idx + 1] = Mim[i][j][e] - mir[4 * e];
                        om[3 * blk * 2 + idx] = Pre[i][j][e] + mir[4 * e + 3]; om[3 * blk * 2 + idx + 1] = Pim[i][j][e] - mir[4 * e + 2];
                    }
                } else {
                    o[idx] = Mre[i][j][e]; o[idx + 1] = Mim[i][j][e];
                    op[idx] = Pre[i][j][e]; op[idx + 1] = Pim[i][j][e];
                }
            }
        }
    if (DUAL) {
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        __syncthreads();
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(s_tmem), "n"(TcRing<DUAL>::TMEM_COLS));
    }
}

// ------------------------------------------------------------------------------------------------ spheroidal rule (NEXT-2)
// eq. (9) in the paper's own coordinates: eta_i Gauss-Laguerre, tau_k Gauss-Legendre, analytic azimuth.
// The weight  W_d(i,k) = w^eta_i w^tau_k (R/2)^3 (eta_i^2 - tau_k^2) e^{-i v cosTh (R/2) eta_i tau_k} (+i)^d J_d(x_ik),
// x_ik = v sinTh (R/2) sqrt((eta_i^2 - 1)(1 - tau_k^2)), does not separate into a ring and an axial factor, so the
// contraction applies it per 8 x 8 sub-tile: the columns (a, q >= 0) are grouped by q and every group is padded to a
// multiple of 8, hence a sub-tile has one q and one q' and needs W_{|q-q'|} (family -) and W_{q+q'} (family +).
// Table layout per position: Wd [ring i][k4-group kc][d = 0..dmax][4 nodes] complex (one TMA bulk copy per stage).

// J_0 .. J_dmax (x), x >= 0: three-term series for x < 1e-3, else Miller's backward recurrence normalised by
// J_0 + 2 sum_{k>=1} J_2k = 1.
__device__ void bessel_j_all(double x, int dmax, double *J) {
    if (x < 1e-3) {
        const double hx = 0.5 * x, h2 = hx * hx;
        double pw = 1.0, fact = 1.0;
        for (int d = 0; d <= dmax; ++d) {
            if (d > 0) { pw *= hx; fact *= d; }
            J[d] = pw / fact * (1.0 - h2 / (d + 1) + h2 * h2 / (2.0 * (d + 1) * (d + 2)));
        }
        return;
    }
    int M = (int)(x + 14.0 * cbrt(x) + 32.0) + dmax;
    M += M & 1;                                              // even start order
    double jp = 0.0, jc = 1e-30, sum = 0.0;                  // J_{k+1}, J_k (unnormalised), k = M
    const double tox = 2.0 / x;
    for (int k = M; k >= 1; --k) {
        const double jm = k * tox * jc - jp;                 // J_{k-1}
        jp = jc; jc = jm;
        if (k - 1 <= dmax) J[k - 1] = jc;
        if (((k - 1) & 1) == 0 && k - 1 > 0) sum += jc;
        if (fabs(jc) > 1e200) { jc *= 1e-200; jp *= 1e-200; sum *= 1e-200; for (int d = k - 1; d <= dmax && d < M; ++d) if (d >= k - 1) J[d] *= 1e-200; }
    }
    const double norm = 1.0 / (2.0 * sum + jc);              // jc = J_0
    for (int d = 0; d <= dmax; ++d) J[d] *= norm;
}

struct TsphArgs {
    PosTabs L; const double *R, *cosT, *sinT, *v; const double *gl_eta, *gl_tau; double eta_scale;
    double *out; double *wd; size_t wd_stride;      // per-position tables (eta_i, tau_k) and weights
    int q0;
};

// grid = (ring, position), block = n_z threads (one per tau node), rounded up to a warp multiple
__global__ void __launch_bounds__(256) k_tpos_sph(const TsphArgs a) {
    const int ring = blockIdx.x, p = blockIdx.y, gp = a.q0 + p;
    const PosTabs &L = a.L;
    double *o = a.out + (size_t)p * L.size();
    const double R = a.R[gp], cT = a.cosT[gp], sT = a.sinT[gp], v = a.v[gp];
    const double s = __dmul_rn(__dmul_rn(0.5, a.eta_scale), R);                      // x = s (eta - 1)
    const double eta = __dadd_rn(1.0, a.gl_eta[ring] / s), weta = a.gl_eta[L.n_rho + ring] / s;
    if (threadIdx.x == 0) o[L.off_rho() + ring] = eta;
    const double hR = __dmul_rn(0.5, R), hR3 = hR * hR * hR;
    cplx *wd = reinterpret_cast<cplx *>(a.wd + (size_t)p * a.wd_stride) + (size_t)ring * L.n_z * (L.dmax + 1);
    for (int k = threadIdx.x; k < L.n_z; k += blockDim.x) {
        const double tau = a.gl_tau[k], wtau = a.gl_tau[L.n_z + k];
        if (ring == 0) o[L.off_zq() + k] = tau;
        const double W = weta * wtau * hR3 * (eta * eta - tau * tau);
        const double x = fabs(v * sT * hR) * sqrt(fmax(0.0, (eta * eta - 1.0) * (1.0 - tau * tau)));
        double sn, cs; sincos(-(v * cT * hR) * (eta * tau), &sn, &cs);
        double J[MAXD + 1];
        bessel_j_all(x, L.dmax, J);
        const bool neg = v * sT < 0.0;                       // J_d(-x) = (-1)^d J_d(x)
        for (int d = 0; d <= L.dmax; ++d) {
            const double j = (neg && (d & 1)) ? -J[d] : J[d];
            // (+i)^d J_d times W e^{-i ...}
            double pr, pi;
            switch (d & 3) { case 0: pr = j; pi = 0.0; break; case 1: pr = 0.0; pi = j; break; case 2: pr = -j; pi = 0.0; break; default: pr = 0.0; pi = -j; }
            const double wr = W * (pr * cs - pi * sn), wi = W * (pr * sn + pi * cs);
            wd[((size_t)(k >> 2) * (L.dmax + 1) + d) * 4 + (k & 3)] = cplx{wr, wi};
        }
    }
}

struct TconSphArgs {
    PosTabs L;
    const double *tabT, *tabP; size_t strideT, strideP;
    const double *wd; size_t wd_stride;
    int nq8T, nq8P;
    const int *qT, *qP;
    const int2 *tiles;
    double *part;                                                // [p][fam 2][prod 3][nq8P][nq8T] complex
    int stages;                                                  // TMA ring depth (2 or 3)
};

constexpr int TS_KCS = 16, TS_STAGE_DOUBLES = TS_KCS * 256;

// grid = (tile, 1, position); 8 warps as 4 (rows) x 2 (cols), warp tile 16 x 32 of a 64 x 64 tile; both families are
// accumulated directly (no ring epilogue): M += (B W_{|q-q'|})^T A, P += (B W_{q+q'})^T A for q, q' > 0.
__global__ void __launch_bounds__(256, 1) k_tcon_sph(const TconSphArgs a) {
    constexpr int NJ = 4;
    extern __shared__ __align__(128) double sm[];
    const int NS = a.stages, nd = a.L.dmax + 1;
    const int w_stage = TS_KCS * nd * 8;                         // doubles of weights per stage
    double *sA = sm, *sB = sA + NS * TS_STAGE_DOUBLES, *sW = sB + NS * TS_STAGE_DOUBLES;
    __shared__ __align__(8) unsigned long long bar[3], empty[3];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, p = blockIdx.z;
    const int2 tl = a.tiles[blockIdx.x];
    const int rt = tl.x, ct = tl.y;
    const int n_rho = a.L.n_rho, nkc = a.L.n_z / 4, spr = (nkc + TS_KCS - 1) / TS_KCS, n_st = n_rho * spr;
    if (tid == 0) { for (int s = 0; s < NS; ++s) { mbar_init(&bar[s], 1); mbar_init(&empty[s], 8); } mbar_fence_init(); }
    __syncthreads();
    const double *gA = a.tabT + (size_t)p * a.strideT + (size_t)ct * n_rho * nkc * 256;
    const double *gB = a.tabP + (size_t)p * a.strideP + (size_t)rt * n_rho * nkc * 256;
    const double *gW = a.wd + (size_t)p * a.wd_stride;
    auto issue = [&](int st) {
        const int ring = st / spr, kc0 = (st % spr) * TS_KCS, nk = min(TS_KCS, nkc - kc0), buf = st % NS;
        const unsigned bytes = (unsigned)nk * 256 * 8, wbytes = (unsigned)nk * nd * 64;
        mbar_expect_tx(&bar[buf], 2 * bytes + wbytes);
        tma_bulk_g2s(sA + buf * TS_STAGE_DOUBLES, gA + ((size_t)ring * nkc + kc0) * 256, bytes, &bar[buf]);
        tma_bulk_g2s(sB + buf * TS_STAGE_DOUBLES, gB + ((size_t)ring * nkc + kc0) * 256, bytes, &bar[buf]);
        tma_bulk_g2s(sW + buf * w_stage, gW + ((size_t)ring * nkc + kc0) * nd * 8, wbytes, &bar[buf]);
    };
    if (tid == 0) for (int st = 0; st < min(NS, n_st); ++st) issue(st);

    const int wr = warp / 2, wc = warp % 2, fr = lane >> 2, fk = lane & 3;
    bool need[2][NJ]; int dm[2][NJ], dp[2][NJ];                  // weight offsets (doubles) into a k4-group of sW; dp < 0: family + empty
    bool any_need = false;
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int r8 = rt * 64 + 16 * wr + 8 * i, c8 = ct * 64 + 32 * wc + 8 * j;
            need[i][j] = (r8 < 2 * a.nq8P) && (c8 < 2 * a.nq8T) && !(r8 >= a.nq8P && c8 >= a.nq8T);
            int qp = 0, qq = 0;
            if (need[i][j]) { qp = max(0, a.qP[r8 % a.nq8P]); qq = max(0, a.qT[c8 % a.nq8T]); }
            dm[i][j] = abs(qq - qp) * 8 + 2 * fk;
            dp[i][j] = (qp > 0 && qq > 0) ? (qq + qp) * 8 + 2 * fk : -1;
            any_need |= need[i][j];
        }
    double Mre[2][NJ][2], Mim[2][NJ][2], Pre[2][NJ][2], Pim[2][NJ][2];
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < NJ; ++j)
            #pragma unroll
            for (int e = 0; e < 2; ++e) Mre[i][j][e] = Mim[i][j][e] = Pre[i][j][e] = Pim[i][j][e] = 0.0;

    for (int st = 0; st < n_st; ++st) {
        const int buf = st % NS, kc0 = (st % spr) * TS_KCS, nk = min(TS_KCS, nkc - kc0);
        mbar_wait(&bar[buf], (st / NS) & 1);
        if (any_need) {
            const double *Ab = sA + buf * TS_STAGE_DOUBLES + (NJ * wc) * 32 + lane;
            const double *Bb = sB + buf * TS_STAGE_DOUBLES + (2 * wr) * 32 + lane;
            const double *Wb = sW + buf * w_stage;
            #pragma unroll 2
            for (int kc = 0; kc < nk; ++kc) {
                double af[NJ], bb[2];
                #pragma unroll
                for (int j = 0; j < NJ; ++j) af[j] = Ab[kc * 256 + j * 32];
                #pragma unroll
                for (int i = 0; i < 2; ++i) bb[i] = Bb[kc * 256 + i * 32];
                const double *wk = Wb + kc * nd * 8;
                #pragma unroll
                for (int i = 0; i < 2; ++i)
                    #pragma unroll
                    for (int j = 0; j < NJ; ++j)
                        if (need[i][j]) {
                            const double2 wm = *reinterpret_cast<const double2 *>(wk + dm[i][j]);
                            dmma884(Mre[i][j][0], Mre[i][j][1], bb[i] * wm.x, af[j]);
                            dmma884(Mim[i][j][0], Mim[i][j][1], bb[i] * wm.y, af[j]);
                            if (dp[i][j] >= 0) {
                                const double2 wp = *reinterpret_cast<const double2 *>(wk + dp[i][j]);
                                dmma884(Pre[i][j][0], Pre[i][j][1], bb[i] * wp.x, af[j]);
                                dmma884(Pim[i][j][0], Pim[i][j][1], bb[i] * wp.y, af[j]);
                            }
                        }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[buf]);
        if (tid == 0 && st >= 1 && st - 1 + NS < n_st) {
            mbar_wait(&empty[(st - 1) % NS], ((st - 1) / NS) & 1);
            issue(st - 1 + NS);
        }
    }
    const size_t blk = (size_t)a.nq8P * a.nq8T;
    double *o = a.part + (size_t)p * 6 * blk * 2;
    #pragma unroll
    for (int i = 0; i < 2; ++i)
        #pragma unroll
        for (int j = 0; j < NJ; ++j)
            #pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int gr = rt * 64 + 16 * wr + 8 * i + fr, gc = ct * 64 + 32 * wc + 8 * j + 2 * fk + e;
                if (!need[i][j] || gr >= 2 * a.nq8P || gc >= 2 * a.nq8T) continue;
                if (a.qP[gr % a.nq8P] < 0 || a.qT[gc % a.nq8T] < 0) continue;            // padding column
                const int hr = gr / a.nq8P, ir = gr % a.nq8P, hc = gc / a.nq8T, ic = gc % a.nq8T;
                const int prod = hr ? 2 : (hc ? 1 : 0);
                const size_t idx = ((size_t)prod * blk + (size_t)ir * a.nq8T + ic) * 2;
                o[idx] = Mre[i][j][e]; o[idx + 1] = Mim[i][j][e];
                o[3 * blk * 2 + idx] = Pre[i][j][e]; o[3 * blk * 2 + idx + 1] = Pim[i][j][e];
            }
}

// ------------------------------------------------------------------------------------------------ rotation (a6)
struct TrotChunk { int b0, b1, st0, nst, nrows; };   // radial functions [b0, b1) of centre P, their states, their body rows
struct TrotArgs {
    const double *part; int n_split; int nq8T, nq8P;
    const double *theta;                     // [p] Theta = angle between R and v
    const int *radT, *lT_st, *mT_st;         // per target state: radial function, l, m
    const int *radP, *lP_st, *mP_st;         // per projectile state
    const int *colT, *colP;                  // [n_rad][WP_MAX_L+1] column of (a, |q|)
    const int *colTst;                       // [NT][lmax+1] column of (radial function of target state ia, q), 0 beyond l
    const int *lradP;                        // [n_rad_P] l of each projectile radial function
    const TrotChunk *chunks; const int *rowbase;   // rowbase[b]: first local body row of radial function b inside its chunk
    int NT, NP, lmax, max_rows;
    double *K; double *H;                    // K [p][NP][NT] complex; H [p][N][N] complex (p: window position)
    double *KT; int ht;                      // optional K^T [p][NT][NP]; ht: write the H_PT, H_TP blocks of H^T instead of H
    int tb;                                  // target states per pass through stages 1 and 2
    // block z: evaluated position (fetch == 0): window position sel_pos(sel, q0 + z), integrals part[z];
    //          fetched position (fetch == 1): z = g * n_fetch + lf -> window position g * n_idx + n_pre + lf,
    //          integrals in stash slot g * n_st + slot0 + lf
    SelDev sel; int q0, fetch, n_fetch, n_st, slot0; const double *stash;
};

// Wigner d^l_{m' m}(beta) = <l m'| e^{-i beta J_y} |l m>, Wigner's sum formula; cb = cos(beta/2), sb = sin(beta/2).
__device__ __forceinline__ double ipow(double x, int n) {        // x^n, n >= 0, by repeated squaring
    double r = 1.0;
    while (n) { if (n & 1) r *= x; x *= x; n >>= 1; }
    return r;
}
__device__ double wigner_d(int l, int mp, int m, double cb, double sb) {
    double tot = 0.0;
    const double num = sqrt(c_fact[l + m] * c_fact[l - m] * c_fact[l + mp] * c_fact[l - mp]);
    for (int k = max(0, m - mp); k <= min(l + m, l - mp); ++k) {
        const double den = c_fact[l + m - k] * c_fact[k] * c_fact[l - k - mp] * c_fact[k - m + mp];
        double term = num / den * ipow(cb, 2 * l - 2 * k + m - mp) * ipow(sb, 2 * k - m + mp);
        tot += ((k - m + mp) & 1) ? -term : term;
    }
    return tot;
}

// grid = (chunk of projectile radial functions, 1, position); block 256.  A CTA handles every product of its chunk in turn
// (S_PT -> K and K^T, H_PT, H_TP), so that the Wigner matrices and the index tables are set up once.  The body-frame rows
// the chunk needs (both families, ring splits summed in order) are staged in shared memory with coalesced loads; then one
// thread per lab-frame output element (beta, alpha), eq. (8):
//   X_lab[beta, alpha] = sum_{q', q} d^{l_b}_{m_b q'}(Theta) d^{l_a}_{m_a q}(Theta) X_body[(b, q'), (a, q)],
// where the signed body-frame element comes from the two q >= 0 families of the contraction:
//   family (-) (weights Phi_{|q-q'|}) when q, q' have the same sign or one is 0, family (+) (Phi_{q+q'}) otherwise,
//   times (-1)^q for q < 0 and (-1)^q' for q' < 0.
__global__ void __launch_bounds__(256) k_trot(const TrotArgs a) {
    extern __shared__ __align__(16) double sd[];     // [lmax+1][W][W] Wigner d, W = 2 lmax + 1; then body rows [2][max_rows][nq8T] complex
    const int tid = threadIdx.x, L = a.lmax, W = 2 * L + 1;
    const TrotChunk ch = a.chunks[blockIdx.x];
    int p; const double2 *part;              // window position (geometry, outputs) and its body-frame integrals
    {
        const size_t per_pos = (size_t)a.n_split * 6 * a.nq8P * a.nq8T;
        if (!a.fetch) { p = sel_pos(a.sel, a.q0 + blockIdx.z); part = reinterpret_cast<const double2 *>(a.part) + blockIdx.z * per_pos; }
        else {
            const int zz = a.q0 + blockIdx.z, g = zz / a.n_fetch, lf = zz - g * a.n_fetch;
            p = g * a.sel.n_idx + a.sel.n_pre + lf;
            part = reinterpret_cast<const double2 *>(a.stash) + ((size_t)g * a.n_st + a.slot0 + lf) * per_pos;
        }
    }
    const int nd = ((L + 1) * W * W + 1) & ~1;
    double2 *body = reinterpret_cast<double2 *>(sd + nd);
    const int nq8T = a.nq8T, NT = a.NT;
    const size_t blk = (size_t)a.nq8P * nq8T, fam_stride = (size_t)a.max_rows * nq8T;
    const int TB = a.tb;                                                          // target states per pass (NT unless shared memory is short)
    double2 *Ep = body + 2 * fam_stride, *Em = Ep + (size_t)a.max_rows * TB;      // [rows][TB] each
    int *s_colT = reinterpret_cast<int *>(Em + (size_t)a.max_rows * TB);          // [NT][L+1] column of (a, q) per target state
    // stage the rows (b, q'), b in [b0, b1), q' = 0..l_b: local row = rowbase[b] + q'
    __shared__ int s_rowsrc[256], s_rowp[256];       // body row (column index of centre P) and q' of each local row
    for (int b = ch.b0 + tid; b < ch.b1; b += blockDim.x)
        for (int r = 0; r <= a.lradP[b]; ++r) { s_rowsrc[a.rowbase[b] + r] = a.colP[b * (WP_MAX_L + 1) + r]; s_rowp[a.rowbase[b] + r] = r; }
    for (int e = tid; e < NT * (L + 1); e += blockDim.x) s_colT[e] = a.colTst[e];
    {
        double sb, cb; sincos(0.5 * a.theta[p], &sb, &cb);
        for (int e = tid; e < (L + 1) * W * W; e += blockDim.x) {
            const int l = e / (W * W), mp = (e / W) % W - L, m = e % W - L;
            sd[e] = (abs(mp) <= l && abs(m) <= l) ? wigner_d(l, mp, m, cb, sb) : 0.0;
        }
    }
    const int NP = a.NP, N = NT + NP;
    const int per_fam = ch.nrows * nq8T;
    // outputs in turn: 0 S_PT -> K, 3 S_PT -> K^T (same staged rows and stage 1 as 0; only with a.KT), 1 H_PT, 2 H_TP
    for (int oi = 0; oi < 4; ++oi) {
        const int yid = (oi == 0) ? 0 : (oi == 1 ? 3 : oi - 1), prod = yid == 3 ? 0 : yid;
        if (yid == 3 && !a.KT) continue;
        __syncthreads();                             // tables ready / the previous output is done with body, Ep, Em
        if (yid != 3) {
            const double2 *src0 = part + (size_t)prod * blk;
            if (a.n_split == 1) {
                // four independent 16-byte loads in flight per thread
                for (int e0 = tid; e0 < 2 * per_fam; e0 += 4 * 256) {
                    double2 v[4]; int dst[4];
                    #pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int e = e0 + 256 * u;
                        dst[u] = -1;
                        if (e < 2 * per_fam) {
                            const int fam = e >= per_fam, r2 = e - fam * per_fam, r = r2 / nq8T, c = r2 - r * nq8T;
                            v[u] = src0[(size_t)fam * 3 * blk + (size_t)s_rowsrc[r] * nq8T + c];
                            dst[u] = fam * (int)fam_stride + r * nq8T + c;
                        }
                    }
                    #pragma unroll
                    for (int u = 0; u < 4; ++u) if (dst[u] >= 0) body[dst[u]] = v[u];
                }
            } else {
                for (int e = tid; e < 2 * per_fam; e += blockDim.x) {
                    const int fam = e >= per_fam, r2 = e - fam * per_fam, r = r2 / nq8T, c = r2 - r * nq8T;
                    const double2 *src = src0 + (size_t)fam * 3 * blk + (size_t)s_rowsrc[r] * nq8T + c;
                    double2 v = {0.0, 0.0};
                    for (int sp = 0; sp < a.n_split; ++sp) { const double2 x = src[(size_t)sp * 6 * blk]; v.x += x.x; v.y += x.y; }
                    body[fam * fam_stride + (size_t)r * nq8T + c] = v;
                }
            }
            __syncthreads();
        }
        // stage 1: contract the target-side index.  For body row (b, p = |q'|) and target state alpha = (a, m_a):
        //   P0 = sum_{q>=0} d^{l_a}_{m_a,q} F0[q],  M0 = sum_{q>0} (-1)^q d_{m_a,-q} F0[q],  P1, M1 the same with family (+),
        //   E+ = P0 + (p == 0 ? M0 : M1)            (q' = +p),      E- = (-1)^p (d_{m_a,0} F0[0] + P1 + M0)   (q' = -p < 0)
        // (with all target states in one pass, output 3 reuses E+, E- of output 0)
        for (int ia0 = 0; ia0 < NT; ia0 += TB) {
            const int tbn = min(TB, NT - ia0);
            if (!(yid == 3 && TB >= NT)) {
                if (ia0) __syncthreads();                                 // the previous pass is done with Ep, Em
                for (int e = tid; e < ch.nrows * tbn; e += blockDim.x) {
                    const int r = e / tbn, ia = ia0 + (e - r * tbn), pq = s_rowp[r];
                    const int la = a.lT_st[ia], ma = a.mT_st[ia];
                    const double *dA = sd + (la * W + ma + L) * W + L;
                    const double2 *f0 = body + (size_t)r * nq8T, *f1 = f0 + fam_stride;
                    const int *ct = s_colT + ia * (L + 1);
                    const double2 x00 = f0[ct[0]];
                    const double d0 = dA[0];
                    double2 P0 = {d0 * x00.x, d0 * x00.y}, M0 = {0.0, 0.0}, P1 = {0.0, 0.0}, M1 = {0.0, 0.0};
                    const double2 Z0 = P0;
                    for (int q = 1; q <= la; ++q) {
                        const int c = ct[q];
                        const double dp = dA[q], dm = (q & 1) ? -dA[-q] : dA[-q];
                        const double2 x0 = f0[c], x1 = f1[c];
                        P0.x += dp * x0.x; P0.y += dp * x0.y; M0.x += dm * x0.x; M0.y += dm * x0.y;
                        P1.x += dp * x1.x; P1.y += dp * x1.y; M1.x += dm * x1.x; M1.y += dm * x1.y;
                    }
                    const double2 mm = (pq == 0) ? M0 : M1;
                    const double sg = (pq & 1) ? -1.0 : 1.0;
                    Ep[e] = {P0.x + mm.x, P0.y + mm.y};
                    Em[e] = {sg * (Z0.x + P1.x + M0.x), sg * (Z0.y + P1.y + M0.y)};
                }
                __syncthreads();
            }
            // stage 2: contract the projectile-side index
            for (int e = tid; e < ch.nst * tbn; e += blockDim.x) {
                // loop order = the order of the output rows (coalesced stores): K and H_PT row-major in (beta, alpha), H_TP and K^T in
                // (alpha, beta); with a.ht the H blocks are written transposed (H^T is what the RK4 sweep streams), so the two swap
                const bool beta_major = (yid == 0) || (yid == 1 && !a.ht) || (yid == 2 && a.ht);
                const int ibl = beta_major ? e / tbn : e % ch.nst, ial = beta_major ? e % tbn : e / ch.nst, ia = ia0 + ial;
                const int ib = ch.st0 + ibl;
                const int rb = a.radP[ib], lb = a.lP_st[ib], mb = a.mP_st[ib];
                const double *dB = sd + (lb * W + mb + L) * W + L;
                const double2 *ep = Ep + (size_t)a.rowbase[rb] * tbn + ial, *em = Em + (size_t)a.rowbase[rb] * tbn + ial;
                double sr = dB[0] * ep[0].x, si = dB[0] * ep[0].y;
                for (int pq = 1; pq <= lb; ++pq) {
                    const double2 xp = ep[pq * tbn], xm = em[pq * tbn];
                    sr += dB[pq] * xp.x + dB[-pq] * xm.x; si += dB[pq] * xp.y + dB[-pq] * xm.y;
                }
                double *o;
                if (yid == 0) o = a.K + (((size_t)p * NP + ib) * NT + ia) * 2;
                else if (yid == 3) o = a.KT + (((size_t)p * NT + ia) * NP + ib) * 2;
                else if (yid == 1) o = a.H + (a.ht ? ((size_t)p * N + ia) * N + NT + ib : ((size_t)p * N + NT + ib) * N + ia) * 2;             // H_PT
                else { o = a.H + (a.ht ? ((size_t)p * N + NT + ib) * N + ia : ((size_t)p * N + ia) * N + NT + ib) * 2; si = -si; }            // H_TP = conj(rot Tb)^T
                *reinterpret_cast<double2 *>(o) = make_double2(sr, si);
            }
            if (yid == 3 && TB < NT) __syncthreads();
        }
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------- host side
struct TransferPlan {
    PosTabs L; int nq8[2], ntile[2]; size_t stride[2]; size_t part_per_pos; int n_split; std::vector<int2> tiles;
    size_t wd_stride = 0;                    // spheroidal rule: doubles of weights W_d(i,k) per position
    size_t per_pos_bytes() const { return ((size_t)L.size() + stride[0] + stride[1] + wd_stride) * 8 + part_per_pos * 8 + 64; }
};

// Columns (a, q >= 0) of a centre, grouped by q.  pad8 (spheroidal rule): every q-group starts at a multiple of 8, so that
// an 8-column block of the contraction has a single q.  Returns the padded column count (a multiple of 8).
static int column_map(const CentreTab &C, bool pad8, std::vector<int> *col_of /*[n_rad][WP_MAX_L+1] or null*/, std::vector<int> *q_of /*[cols] or null*/) {
    int col = 0;
    if (col_of) col_of->assign((size_t)C.n_rad * (WP_MAX_L + 1), -1);
    std::vector<int> q;
    for (int qq = 0; qq <= C.l_max; ++qq) {
        if (pad8) while (col & 7) { q.push_back(-1); ++col; }
        for (int a = 0; a < C.n_rad; ++a) if (C.l[a] >= qq) { if (col_of) (*col_of)[(size_t)a * (WP_MAX_L + 1) + qq] = col; q.push_back(qq); ++col; }
    }
    while (col & 7) { q.push_back(-1); ++col; }
    if (q_of) *q_of = q;
    return col;
}

static TransferPlan make_plan(const wpccc_basis *B, int n_split) {
    TransferPlan P;
    const bool sph = B->quad.kind == 1;
    P.L.n_rho = B->quad.n_rho; P.L.n_z = B->quad.n_z; P.L.n_phi = B->quad.n_phi; P.L.dmax = B->c[0].l_max + B->c[1].l_max;
    if (sph) P.wd_stride = (size_t)P.L.n_rho * P.L.n_z * (P.L.dmax + 1) * 2;
    for (int s = 0; s < 2; ++s) {
        P.nq8[s] = column_map(B->c[s], sph, nullptr, nullptr);
        P.ntile[s] = (2 * P.nq8[s] + 63) / 64;
        P.stride[s] = (size_t)P.ntile[s] * 64 * P.L.n_rho * P.L.n_z;
    }
    P.n_split = n_split;
    P.part_per_pos = (size_t)n_split * 6 * P.nq8[0] * P.nq8[1] * 2;
    for (int rt = 0; rt < P.ntile[1]; ++rt)
        for (int ct = 0; ct < P.ntile[0]; ++ct)
            if (!(rt * 64 >= P.nq8[1] && ct * 64 >= P.nq8[0])) P.tiles.push_back(make_int2(rt, ct));
    return P;
}

// Ring splits (split-K of the contraction) as a function of the positions per launch: none once a launch has two
// waves of CTAs on the 148 SMs; for a handful of positions (wpccc_matrix_elements) enough to occupy the GPU.
static int pick_split(const wpccc_basis *B, int chunk) {
    if (B->quad.kind == 1) return 1;
    TransferPlan P = make_plan(B, 1);
    const long long ctas = (long long)P.tiles.size() * std::max(chunk, 1);
    int s = (int)std::min<long long>((296 + ctas - 1) / ctas, std::max(1, B->quad.n_rho / 4));
    return std::max(1, s);
}

size_t wp_transfer_ws_bytes(const wpccc_basis *B, int n_pos_chunk) {
    TransferPlan P = make_plan(B, pick_split(B, n_pos_chunk));
    return P.per_pos_bytes() * (size_t)n_pos_chunk + P.tiles.size() * sizeof(int2) + 4096 +
           2 * (size_t)(B->c[0].n_rad + B->c[1].n_rad) * (WP_MAX_L + 1) * sizeof(int) +
           2 * (size_t)(P.nq8[0] + P.nq8[1]) * sizeof(int) +
           (size_t)B->c[1].n_rad * (sizeof(TrotChunk) + sizeof(int)) + (size_t)B->c[0].n_states * (WP_MAX_L + 1) * sizeof(int) + 2048;
}

int wp_transfer_chunk_positions(const wpccc_basis *B, size_t ws_bytes) {
    if (wp_transfer_ws_bytes(B, 1) > ws_bytes) return 0;
    int lo = 1, hi = 1 << 16;                       // largest chunk whose workspace fits (bytes grow with the chunk)
    while (lo < hi) { const int mid = (lo + hi + 1) / 2; if (wp_transfer_ws_bytes(B, mid) <= ws_bytes) lo = mid; else hi = mid - 1; }
    return lo;
}

int wp_transfer_default_chunk(const wpccc_basis *B) {
    // a multiple of the SM count (every tile CTA has the same work, so launches are whole waves), node tables <= 17 GB
    // (configs[3]: 113 MB per position: 148 positions = 16.7 GB; halving the chunk leaves a ragged last wave)
    TransferPlan P = make_plan(B, 1);
    const size_t tab = (P.stride[0] + P.stride[1]) * 8;
    int c = 148;
    while (c > 1 && (size_t)c * tab > ((size_t)17 << 30)) c /= 2;
    return c;
}

size_t wp_transfer_stash_doubles(const wpccc_basis *B) { return make_plan(B, 1).part_per_pos; }
static size_t dual_smem_bytes(const TransferPlan &P) {
    return ((size_t)2 * TcRing<true>::STAGES * TcRing<true>::STAGE_DOUBLES + TcRing<true>::ACC_DOUBLES + 2 * P.L.n_z + 2 * (size_t)(P.L.dmax + 2) * P.L.n_rho) * 8;
}
bool wp_transfer_mirror_ok(const wpccc_basis *B) { return B->quad.kind == 0 && dual_smem_bytes(make_plan(B, 1)) <= 226 * 1024; }

int wp_transfer(wpccc_basis *B, int n_pos, const double *d_R, const double *d_cos, const double *d_sin, const double *d_theta,
                const double *d_v, double *d_K, double *d_H, void *ws, size_t ws_bytes, int chunk, cudaStream_t s,
                const TransferSel *sel, double *d_KT) {
    if (n_pos <= 0) return 0;
    SelDev sd{0, 0, 0, 0};
    int n_eval = n_pos, n_fetch = 0;                 // evaluated positions of this call; fetched indices per group
    if (sel) {
        if (n_pos != sel->n_groups * sel->n_idx) WP_FAIL(WPCCC_EINVAL, "transfer: selection does not match the window");
        n_fetch = sel->suf0 - sel->n_pre;
        sd = SelDev{sel->n_idx - n_fetch, sel->n_idx, sel->n_pre, sel->suf0};
        n_eval = sel->n_groups * sd.n_c;
    }
    static PerDevice consts;
    if (wp_raise(consts, 1)) {
        double f[2 * WP_MAX_L + 2]; f[0] = 1.0;
        for (int i = 1; i < 2 * WP_MAX_L + 2; ++i) f[i] = f[i - 1] * i;
        WP_CUDA(cudaMemcpyToSymbol(c_fact, f, sizeof f));
        double tn[NLQ];
        for (int l = 0; l <= WP_MAX_L; ++l) for (int q = 0; q <= l; ++q) tn[lq_index(l, q)] = std::sqrt((2 * l + 1) / 2.0 * f[l - q] / f[l + q]);
        WP_CUDA(cudaMemcpyToSymbol(c_thnorm, tn, sizeof tn));
    }
    const int max_chunk = wp_transfer_chunk_positions(B, ws_bytes);
    if (max_chunk < 1) WP_FAIL(WPCCC_ENOMEM, "transfer workspace too small (%zu bytes)", ws_bytes);
    chunk = std::max(1, std::min(std::min(chunk, max_chunk), std::max(n_eval, 1)));
    const int n_split = sel ? 1 : pick_split(B, chunk);
    TransferPlan P = make_plan(B, n_split);

    // carve the workspace
    char *w = (char *)ws; size_t off = 0;
    auto take = [&](size_t bytes) { off = (off + 255) & ~(size_t)255; void *p = w + off; off += bytes; return p; };
    double *d_pos = (double *)take((size_t)chunk * P.L.size() * 8);
    double *d_tab[2] = {(double *)take((size_t)chunk * P.stride[0] * 8), (double *)take((size_t)chunk * P.stride[1] * 8)};
    double *d_part = (double *)take((size_t)chunk * P.part_per_pos * 8);
    const bool sph = B->quad.kind == 1;
    double *d_wd = sph ? (double *)take((size_t)chunk * P.wd_stride * 8) : nullptr;
    int2 *d_tiles = (int2 *)take(P.tiles.size() * sizeof(int2));
    int *d_colidx[2], *d_qcol[2];
    for (int c = 0; c < 2; ++c) { d_colidx[c] = (int *)take((size_t)B->c[c].n_rad * (WP_MAX_L + 1) * 4); d_qcol[c] = (int *)take((size_t)P.nq8[c] * 4); }
    // rotation chunks: consecutive projectile radial functions whose body rows (both families) fit ~48 KB of shared memory
    const int lmx = std::max(B->c[0].l_max, B->c[1].l_max);
    const size_t rot_nd = (((size_t)(lmx + 1) * (2 * lmx + 1) * (2 * lmx + 1) + 1) & ~(size_t)1) * 8;
    std::vector<TrotChunk> rchunks; std::vector<int> rowbase(B->c[1].n_rad, 0);
    int rot_max_rows = 0;
    {
        const CentreTab &C = B->c[1];
        const size_t rot_fixed = rot_nd + (size_t)B->c[0].n_states * (lmx + 1) * 4 + 16;
        // four CTAs per SM hide the staging latency (cfg 1: 36.8 ms at 100 KB, 26.6 ms at 48 KB; cfg 3: 395 ms per batch with
        // one radial function per chunk at 48 KB, 459 ms with 16 body rows per chunk at 100 KB)
        const size_t rot_target = 48 * 1024;
        const int cap = std::min(256, std::max(C.l_max + 1, (int)((rot_target > rot_fixed ? rot_target - rot_fixed : 0) / (2 * ((size_t)P.nq8[0] + B->c[0].n_states) * 16))));
        TrotChunk cur{0, 0, 0, 0, 0};
        for (int b = 0; b < C.n_rad; ++b) {
            if (cur.nrows + C.l[b] + 1 > cap) { rchunks.push_back(cur); cur = TrotChunk{b, b, C.rad_first[b], 0, 0}; }
            rowbase[b] = cur.nrows; cur.nrows += C.l[b] + 1; cur.nst += 2 * C.l[b] + 1; cur.b1 = b + 1;
        }
        rchunks.push_back(cur);
        for (auto &c : rchunks) rot_max_rows = std::max(rot_max_rows, c.nrows);
    }
    TrotChunk *d_rchunks = (TrotChunk *)take(rchunks.size() * sizeof(TrotChunk));
    int *d_rowbase = (int *)take(rowbase.size() * sizeof(int));
    int *d_colTst = (int *)take((size_t)B->c[0].n_states * (lmx + 1) * sizeof(int));
    if (off > ws_bytes) WP_FAIL(WPCCC_ENOMEM, "transfer workspace too small");
    WP_CUDA(cudaMemcpyAsync(d_rchunks, rchunks.data(), rchunks.size() * sizeof(TrotChunk), cudaMemcpyHostToDevice, s));
    WP_CUDA(cudaMemcpyAsync(d_rowbase, rowbase.data(), rowbase.size() * sizeof(int), cudaMemcpyHostToDevice, s));
    // stages 1 and 2 of the rotation work on all N_T target states at once, or in passes of rot_tb states when the intermediate
    // [rows][N_T] arrays would not fit (wide bases: the paper's two-centre l_max = 5, N_T = 955)
    const size_t rot_base = rot_nd + 2 * (size_t)rot_max_rows * P.nq8[0] * 16 + (size_t)B->c[0].n_states * (lmx + 1) * 4 + 16;
    int rot_tb = B->c[0].n_states;
    while (rot_tb > 32 && rot_base + 2 * (size_t)rot_max_rows * rot_tb * 16 > 200 * 1024) rot_tb = (rot_tb + 1) / 2;
    const size_t rot_smem = rot_base + 2 * (size_t)rot_max_rows * rot_tb * 16;
    if (rot_smem > 220 * 1024) WP_FAIL(WPCCC_EINVAL, "transfer: basis too large for the rotation kernel's shared memory");
    static PerDevice rot_attr;
    if (wp_raise(rot_attr, rot_smem)) WP_CUDA(cudaFuncSetAttribute(k_trot, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rot_smem));
    {   // padding columns of the node tables are never written by k_ttab: zero the buffer once per API call
        const size_t tab_bytes = (size_t)((char *)d_part - (char *)d_tab[0]);
        if (B->tab_zeroed != d_tab[0] || B->tab_zeroed_bytes != tab_bytes) {      // (the layout depends on the chunk size)
            WP_CUDA(cudaMemsetAsync(d_tab[0], 0, tab_bytes, s));
            B->tab_zeroed = d_tab[0]; B->tab_zeroed_bytes = tab_bytes;
        }
    }
    WP_CUDA(cudaMemcpyAsync(d_tiles, P.tiles.data(), P.tiles.size() * sizeof(int2), cudaMemcpyHostToDevice, s));
    std::vector<int> hcol[2], hq[2];
    for (int c = 0; c < 2; ++c) {
        column_map(B->c[c], sph, &hcol[c], &hq[c]);
        WP_CUDA(cudaMemcpyAsync(d_colidx[c], hcol[c].data(), hcol[c].size() * 4, cudaMemcpyHostToDevice, s));
        WP_CUDA(cudaMemcpyAsync(d_qcol[c], hq[c].data(), hq[c].size() * 4, cudaMemcpyHostToDevice, s));
    }

    // node-table kernel configuration: 64 z' nodes per CTA when n_z allows (n_z is a multiple of 16)
    const int nlq = (lmx + 1) * (lmx + 2) / 2;
    const int KC = (P.L.n_z % 64 == 0) ? 64 : ((P.L.n_z % 32 == 0) ? 32 : 16);
    const size_t tab_smem = (size_t)(7 + nlq) * KC * 8 + (size_t)KC * 4 + 64;
    static PerDevice con_attr, dual_attr;
    const size_t con_tabs = 2 * P.L.n_z + 2 * (size_t)(P.L.dmax + 2) * P.L.n_rho;
    const size_t con_smem = ((size_t)2 * TcRing<false>::STAGES * TcRing<false>::STAGE_DOUBLES + con_tabs) * 8;
    const size_t dual_smem = dual_smem_bytes(P);
    if (!sph && con_smem > 220 * 1024) WP_FAIL(WPCCC_EINVAL, "transfer: quadrature too large for the contraction kernel's shared memory");
    // spheroidal contraction: ring of operand stages + the weights of each stage
    const int sph_nd = P.L.dmax + 1;
    const int sph_stages = (3 * ((size_t)2 * TS_STAGE_DOUBLES * 8 + (size_t)TS_KCS * sph_nd * 64) <= 226 * 1024) ? 3 : 2;
    const size_t sph_smem = (size_t)sph_stages * ((size_t)2 * TS_STAGE_DOUBLES * 8 + (size_t)TS_KCS * sph_nd * 64);
    static PerDevice sph_attr;
    if (sph && wp_raise(sph_attr, sph_smem)) WP_CUDA(cudaFuncSetAttribute(k_tcon_sph, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sph_smem));
    // mirror-pair kernel: whenever some evaluated position of this window has a stash slot
    const bool dual = sel && sel->stash && sel->n_st > 0 && sel->i0 < sel->i_mid && sel->i0 + sel->n_pre > sel->i_mid - sel->n_st;
    if (dual && dual_smem > 226 * 1024) WP_FAIL(WPCCC_EINVAL, "transfer: mirror stash requested but the pair kernel does not fit shared memory");
    if (!sph && wp_raise(con_attr, con_smem)) WP_CUDA(cudaFuncSetAttribute(k_tcon<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)con_smem));
    if (dual && wp_raise(dual_attr, dual_smem)) WP_CUDA(cudaFuncSetAttribute(k_tcon<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dual_smem));

    const int NT = B->c[0].n_states, NP = B->c[1].n_states, N = NT + NP;
    {   // column of (radial function of target state ia, q) for q <= l, position-independent
        std::vector<int> cst((size_t)NT * (lmx + 1), 0);
        for (int ia = 0; ia < NT; ++ia)
            for (int q = 0; q <= B->c[0].st_l[ia]; ++q) cst[(size_t)ia * (lmx + 1) + q] = hcol[0][(size_t)B->c[0].st_rad[ia] * (WP_MAX_L + 1) + q];
        WP_CUDA(cudaMemcpyAsync(d_colTst, cst.data(), cst.size() * 4, cudaMemcpyHostToDevice, s));
    }
    TrotArgs tr{}; tr.n_split = n_split; tr.nq8T = P.nq8[0]; tr.nq8P = P.nq8[1]; tr.theta = d_theta;
    tr.radT = B->c[0].d_st_rad; tr.lT_st = B->c[0].d_st_l; tr.mT_st = B->c[0].d_st_m;
    tr.radP = B->c[1].d_st_rad; tr.lP_st = B->c[1].d_st_l; tr.mP_st = B->c[1].d_st_m;
    tr.colT = d_colidx[0]; tr.colP = d_colidx[1]; tr.colTst = d_colTst; tr.NT = NT; tr.NP = NP;
    tr.lmax = lmx; tr.K = d_K; tr.H = d_H; tr.KT = d_KT; tr.ht = d_KT != nullptr;
    tr.lradP = B->c[1].d_l; tr.chunks = d_rchunks; tr.rowbase = d_rowbase; tr.max_rows = rot_max_rows;
    tr.sel = sd; tr.tb = rot_tb;
    for (int p0 = 0; p0 < n_eval; p0 += chunk) {
        const int np = std::min(chunk, n_eval - p0);
        TposArgs ta{}; ta.L = P.L; ta.R = d_R; ta.cosT = d_cos; ta.sinT = d_sin; ta.v = d_v; ta.sel = sd; ta.q0 = p0;
        ta.gl_rho = B->d_gl_rho; ta.gl_phi = B->d_gl_phi; ta.gl_zq = B->d_gl_zq; ta.gl_zh = B->d_gl_zh;
        ta.rho_max = B->quad.rho_max; ta.z_pad = B->quad.z_pad; ta.phi_rule = B->quad.phi_rule; ta.out = d_pos;
        wp_span_begin(B, FAM_TTAB, s);
        if (sph) {
            TsphArgs ts{}; ts.L = P.L; ts.R = d_R; ts.cosT = d_cos; ts.sinT = d_sin; ts.v = d_v; ts.gl_eta = B->d_gl_rho; ts.gl_tau = B->d_gl_zh;
            ts.eta_scale = B->quad.eta_scale; ts.out = d_pos; ts.wd = d_wd; ts.wd_stride = P.wd_stride; ts.q0 = p0;
            k_tpos_sph<<<dim3(P.L.n_rho, np), std::min(256, (P.L.n_z + 31) / 32 * 32), 0, s>>>(ts);
        } else k_tpos<<<np, 128, 0, s>>>(ta);
        TtabArgs tb{}; tb.L = P.L; tb.pos = d_pos; tb.R = d_R; tb.sel = sd; tb.q0 = p0; tb.h = B->h; tb.Nr = B->Nr; tb.KC = KC; tb.sph = sph; tb.rgrid = B->d_rgrid;
        for (int c = 0; c < 2; ++c) {
            tb.Ut[c] = B->c[c].d_Ut; tb.lrad[c] = B->c[c].d_l; tb.n_rad[c] = B->c[c].n_rad; tb.nf_pad[c] = B->c[c].nf_pad;
            tb.nq8[c] = P.nq8[c]; tb.ntile[c] = P.ntile[c]; tb.colidx[c] = d_colidx[c]; tb.out[c] = d_tab[c]; tb.pos_stride[c] = P.stride[c];
            tb.lmax[c] = B->c[c].l_max;
        }
        tb.Zother[0] = B->c[1].Z; tb.Zother[1] = B->c[0].Z;
        dim3 gt(P.L.n_rho * (P.L.n_z / KC), 2, np);
        k_ttab<<<gt, 256, tab_smem, s>>>(tb);
        wp_span_end(B, s, 2);
        B->units[FAM_TTAB] += np;
        WP_CUDA(cudaGetLastError());

        TconArgs tc{}; tc.L = P.L; tc.pos = d_pos; tc.tabT = d_tab[0]; tc.tabP = d_tab[1]; tc.strideT = P.stride[0]; tc.strideP = P.stride[1];
        tc.nq8T = P.nq8[0]; tc.nq8P = P.nq8[1]; tc.ntT = P.ntile[0]; tc.ntP = P.ntile[1]; tc.qT = d_qcol[0]; tc.qP = d_qcol[1];
        tc.tiles = d_tiles; tc.n_tiles = (int)P.tiles.size(); tc.n_split = n_split; tc.part = d_part;
        tc.sel = sd; tc.q0 = p0;
        if (dual) { tc.n_st = sel->n_st; tc.i0 = sel->i0; tc.i_mid = sel->i_mid; tc.stash = sel->stash; }
        dim3 gc((unsigned)P.tiles.size(), n_split, np);
        wp_span_begin(B, FAM_TCON, s);
        if (sph) {
            TconSphArgs th{}; th.L = P.L; th.tabT = d_tab[0]; th.tabP = d_tab[1]; th.strideT = P.stride[0]; th.strideP = P.stride[1];
            th.wd = d_wd; th.wd_stride = P.wd_stride; th.nq8T = P.nq8[0]; th.nq8P = P.nq8[1]; th.qT = d_qcol[0]; th.qP = d_qcol[1];
            th.tiles = d_tiles; th.part = d_part; th.stages = sph_stages;
            k_tcon_sph<<<gc, 256, sph_smem, s>>>(th);
        } else if (dual) k_tcon<4, true><<<gc, 256, dual_smem, s>>>(tc);
        else k_tcon<4, false><<<gc, 256, con_smem, s>>>(tc);
        wp_span_end(B, s, 1);
        B->units[FAM_TCON] += np;
        WP_CUDA(cudaGetLastError());

        tr.part = d_part; tr.q0 = p0; tr.fetch = 0;
        wp_span_begin(B, FAM_ROT, s);
        k_trot<<<dim3((unsigned)rchunks.size(), 1, np), 256, rot_smem, s>>>(tr);
        wp_span_end(B, s, 1);
        B->units[FAM_ROT] += np;
        WP_CUDA(cudaGetLastError());
    }
    if (n_fetch > 0) {       // positions whose integrals an earlier window left in the stash
        tr.part = nullptr; tr.q0 = 0; tr.fetch = 1; tr.n_fetch = n_fetch; tr.n_st = sel->n_st; tr.stash = sel->stash;
        tr.slot0 = (int)(sel->i0 + sel->n_pre - sel->i_mid - 1);
        const int total = sel->n_groups * n_fetch;
        for (int z0 = 0; z0 < total; z0 += 32768) {
            tr.q0 = z0;                      // fetch mode: first (g, lf) pair of this launch
            wp_span_begin(B, FAM_ROT, s);
            k_trot<<<dim3((unsigned)rchunks.size(), 1, (unsigned)std::min(32768, total - z0)), 256, rot_smem, s>>>(tr);
            wp_span_end(B, s, 1);
            WP_CUDA(cudaGetLastError());
        }
        B->units[FAM_ROT] += total;
    }
    return 0;
}
