// Internal declarations shared by the translation units of libwpccc.so (not part of the C ABI).
// Notation follows the paper (arXiv 2403.04252) and DESIGN.md: centres T, P; radial functions a, a';
// states alpha = (a, m); multipole lambda; F^c_lambda(a',a;R) radial entries of eq. (7); D^T, D^P of eq. (6);
// body-frame two-centre integrals of eq. (9) rotated by Wigner d(Theta) as in eq. (8).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "wpccc.h"

#define WP_MAX_L 10       // largest orbital momentum supported per centre
#define WP_MAX_LAMBDA 20  // largest multipole (2 * WP_MAX_L)
#define WP_NFAM 8         // timing families (wpccc_last_timing)
#define WP_SCRATCH_BYTES (1u << 20)   // index scratch of wpccc_probabilities inside the basis arena

enum { FAM_GEMM = 0, FAM_DASM = 1, FAM_TTAB = 2, FAM_TCON = 3, FAM_ROT = 4, FAM_FACT = 5, FAM_SWEEP = 6, FAM_OTHER = 7 };

void wp_set_error(const char *fmt, ...);
#define WP_FAIL(code, ...) do { wp_set_error(__VA_ARGS__); return (code); } while (0)
#define WP_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
    wp_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); return WPCCC_ECUDA; } } while (0)

// Row of a buffer for position p of a launch: p = g * n + li  ->  g * ld + fold(off + li), where fold(i) = i for
// i <= mid and mid2 - i beyond (the mirror position (b, -z) of a z-grid symmetric about 0); n == 0: identity.
struct PosMap { int n, ld, off, mid2; };    // mid2 < 0: no folding
__host__ __device__ inline size_t pos_row(const PosMap &m, int p) {
    if (m.n == 0) return (size_t)p;
    const int g = p / m.n;
    int i = m.off + (p - g * m.n);
    if (m.mid2 >= 0 && 2 * i > m.mid2) i = m.mid2 - i;
    return (size_t)g * m.ld + i;
}

// Mirror pairs of a z-grid symmetric about 0 (two-centre propagation).  The body-frame integrals of eq. (9) at (b, -z)
// and (b, +z) share R, the quadrature nodes, the node tables and the ring weights Phi_Delta(v rho' sinTheta); only the
// axial phase e^{-i v cosTheta (z' - R/2)} is complex-conjugated.  A window of wpccc_propagate therefore evaluates
// the integrals only at the positions selected here and, for those with a free stash slot, also writes the
// integrals of the mirror position, which a later window fetches instead of recomputing them.
// Window position p = g * n_idx + li (half-step index i = i0 + li); evaluated li: [0, n_pre) and [suf0, n_idx),
// fetched li: [n_pre, suf0), i.e. the indices in (i_mid, i_mid + n_st].  Stash slot of (g, i): g * n_st + i - i_mid - 1.
struct TransferSel {
    int n_groups, n_idx, n_pre, suf0;
    long long i0, i_mid;
    int n_st;                    // stash depth (half-step indices per group)
    double *stash;               // [n_groups * n_st] slots of wp_transfer_stash_doubles(B) doubles
};

// One n-tile of the grouped direct GEMM: columns [n0, n0+cnt) of multipole `lam` of centre `c`.
struct GemmTile { int c, lam, n0, cnt; };

// Column of the transfer node tables: radial function `rad` with body-frame projection q >= 0.
struct CentreTab {
    double Z = 0;
    int n_rad = 0, n_states = 0, l_max = 0;
    std::vector<int> l, kind, nq;
    std::vector<double> eps;
    std::vector<int> st_rad, st_l, st_m, rad_first;
    // direct: entries e = (a' <= a, lambda), grouped by lambda
    int n_pairs = 0, E = 0;
    std::vector<int> lam_off, ent_a1, ent_a, ent_lam, ent_pair;
    // transfer: columns (a, q >= 0), grouped by q
    int nqc = 0, nqc_pad = 0;
    std::vector<int> col_rad, col_q, q_off;
    // device tables (inside the caller's arena)
    double *d_PP = nullptr;        // [n_pairs][Kpad]  w_k u_a'(r_k) u_a(r_k), k = 1..Nr (index k-1), zero padded
    int    *d_ent_pair = nullptr;  // [E]              pair row of entry e
    int    *d_ent_lookup = nullptr;// [lambda_max+1][n_rad][n_rad]  entry index of (lambda, a', a), -1 if not allowed
    int    *d_pair_off = nullptr;  // [n_pairs+1]      first slot of pair (a' <= a) in the pair-major copy of F (slots: lambda ascending)
    int    *d_ent_perm = nullptr;  // [E]              pair-major slot of entry e
    int    *d_st_pack = nullptr;   // [n_states]       rad | l << 16 | (l*l + l + m) << 20
    std::vector<int> pair_off, ent_perm, st_pack;
    double *d_G = nullptr;         // [(Lc+1)^2][(Lc+1)^2][lambda_max+1]  G^lambda_{(l'm'),(lm)} of eq. (6)
    double *d_Ut = nullptr;        // [Nr+1][nf_pad]   row k: pairs (u_a(r_k), g_a(r_k)), a = 0..n_rad-1
    int    *d_st_rad = nullptr, *d_st_l = nullptr, *d_st_m = nullptr;   // [n_states]
    double *d_eps = nullptr;       // [n_rad]
    int    *d_l = nullptr;         // [n_rad]
    int    *d_col_rad = nullptr, *d_col_q = nullptr;                    // [nqc_pad] (-1 padding)
    int    *d_rad_first = nullptr; // [n_rad]
    int nf_pad = 0;
};

struct wpccc_basis {
    int n_centres = 0, Nr = 0, Kpad = 0, lambda_max = 0, n_tot = 0;
    double h = 0, Z_proj = 0;
    wpccc_quad quad{};
    bool has_quad = false;
    CentreTab c[2];
    int E_tot = 0;
    std::vector<GemmTile> tiles;
    // shared device tables
    double *d_rp = nullptr;    // [lambda_max+1][Kpad] r_k^lambda
    double *d_rm = nullptr;    // [lambda_max+1][Kpad] r_k^-(lambda+1)
    double *d_rk = nullptr;    // [Kpad] r_k (0 in the padding)
    double *d_rgrid = nullptr; // [Nr+1] r_0 = 0 .. r_Nr of a non-uniform radial grid (wpccc_setup_basis_grid); nullptr: uniform r_k = k h
    GemmTile *d_tiles = nullptr;
    int *d_ent_lam = nullptr;   // [E_tot] multipole of every radial entry (both centres)
    double2 *d_dtab = nullptr;  // [Nr+1][E_tot] (P_e[g], Q_e[g]) prefix/suffix sums of eq. (7), caller-owned; nullptr: GEMM
    double *d_gl_rho = nullptr, *d_gl_phi = nullptr, *d_gl_zq = nullptr, *d_gl_zh = nullptr;  // GL x,w on [-1,1]: [2][n]
    int    *d_st_rad_glob = nullptr;  // [n_tot] global radial-function index of every state (centre T functions first)
    int    *d_rad_info = nullptr;     // [n_rad_tot] 2 * centre + kind (0 bound, 1 wave packet) of every radial function
    char   *d_scratch = nullptr;      // WP_SCRATCH_BYTES of index scratch for wpccc_probabilities (sorted order, b)
    int n_rad_tot = 0;
    char *arena = nullptr; size_t arena_bytes = 0;
    const void *tab_zeroed = nullptr; size_t tab_zeroed_bytes = 0;   // node-table buffer whose padding columns are zero (per API call)
    // timing
    cudaStream_t side = nullptr;   // element kernels of wpccc_propagate
    cudaStream_t hi = nullptr;     // RK4 sweep of wpccc_propagate (highest priority: few CTAs, on the critical path)
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_join2 = nullptr;
    std::vector<cudaEvent_t> ev_pool;
    struct Span { int fam; cudaEvent_t a, b; };
    std::vector<Span> spans;
    size_t ev_used = 0;
    double last_ms[WP_NFAM] = {0};
    long long last_launches[WP_NFAM] = {0};
    long long launches[WP_NFAM] = {0};
    long long groups[WP_NFAM] = {0};
    long long units[WP_NFAM] = {0};       // positions processed per family in the last call (wpccc_last_units)
    int cur_fam = 0; bool cur_sampled = false;
    // options (wpccc_set_option) and the per-trajectory outcome of the last wpccc_propagate (wpccc_last_status)
    struct Options {
        int mirror_pairs = 1;        // evaluate the body-frame integrals of (b, -z), (b, +z) together on symmetric z-grids
        int solve_route = 0;         // 0: Cholesky factor of I - K K^H + triangular solves per RK4 stage; 1: explicit inverse (Gauss-Jordan)
        int inverse_kernel = 0;      // solve_route 1: 0 automatic, 1 shared-memory kernel, 2 global-memory blocked kernel
        int inverse_chunk_cols = 0;  // solve_route 1, register kernel: K staged in chunks of this many columns (0: automatic)
        int sweep_cluster = 0;       // CTAs per trajectory of the two-centre sweep / per unit of the one-centre sweep: 0 automatic, 1, 2, 4 forced
        bool timing = true;          // record CUDA events per kernel family (wpccc_last_timing)
    } opt;
    std::vector<int> last_status;
};

// cudaFuncSetAttribute / constant uploads are per device: remember the largest value set on each device ordinal
struct PerDevice { size_t v[64] = {0}; };
inline bool wp_raise(PerDevice &a, size_t want) {
    int d = 0; cudaGetDevice(&d); d &= 63;
    if (want > a.v[d]) { a.v[d] = want; return true; }
    return false;
}

// timing helpers (api.cu)
void wp_span_begin(wpccc_basis *B, int fam, cudaStream_t s);
void wp_span_end(wpccc_basis *B, cudaStream_t s, int n_launches);
void wp_timing_reset(wpccc_basis *B);

// ---- direct.cu ----
// F[p][off_c + e] for all entries of all centres; R = |R_p|.
// Optional maps: R is read at row pos_row(rmap, p), F written at row pos_row(fmap, p).
int wp_direct_gemm(wpccc_basis *B, int n_pos, const double *d_R, double *d_F, int ldF, cudaStream_t s,
                   const PosMap *rmap = nullptr, const PosMap *fmap = nullptr);
// Real direct blocks without time phase: Dre[p][N_c][N_c] = -charge * sum_lambda sgn^lambda G P_lambda^mu(cos) F.
int wp_direct_assemble(wpccc_basis *B, int c, int n_pos, const double *d_cos, const double *d_F, int ldF,
                       double *d_out, int ld_out, long long pos_stride, int complex_out, cudaStream_t s,
                       const PosMap *fmap = nullptr);   // F of position p is row pos_row(fmap, p)

// ---- transfer.cu ----
size_t wp_transfer_ws_bytes(const wpccc_basis *B, int n_pos_chunk);
int wp_transfer_chunk_positions(const wpccc_basis *B, size_t ws_bytes);
// Lab-frame S_PT -> d_K [p][N_P][N_T]; H_PT -> d_H rows N_T.., cols 0..; H_TP -> d_H rows 0.., cols N_T..  (no time phases).
// `chunk` positions are processed per launch group (node tables of a chunk should stay L2-resident).
// With `sel` (n_pos = sel->n_groups * sel->n_idx) only the selected positions are evaluated (ring splits off) and the
// others come from sel->stash.
int wp_transfer(wpccc_basis *B, int n_pos, const double *d_R, const double *d_cos, const double *d_sin, const double *d_theta,
                const double *d_v, double *d_K, double *d_H, void *ws, size_t ws_bytes, int chunk, cudaStream_t s,
                const TransferSel *sel = nullptr, double *d_KT = nullptr);   // d_KT: also K^T [p][N_T][N_P], and the H_PT / H_TP blocks go to H^T
size_t wp_transfer_stash_doubles(const wpccc_basis *B);   // doubles per stash slot
bool wp_transfer_mirror_ok(const wpccc_basis *B);         // the mirror-pair contraction kernel fits shared memory
int wp_transfer_default_chunk(const wpccc_basis *B);

// ---- sweep.cu ----
// Factorises the overlap system of every position: flags[p] = 0, or 1 zero pivot / 2 |S_PT| >= 1 / 3 not positive definite.
int wp_factor(wpccc_basis *B, int n_pos, const double *d_K, double *d_factor, int *d_flags, void *d_scratch, cudaStream_t s);   // d_factor: wp_factor_elems(N_P) complex per position (sweep.cuh)

// ---- device helpers ----
__host__ __device__ inline int lm_index(int l, int m) { return l * l + l + m; }
