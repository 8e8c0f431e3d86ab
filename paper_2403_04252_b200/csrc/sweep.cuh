// a8: RK4 sweep kernels (Algorithm 1) -- declarations shared by api.cu and sweep.cu.
#pragma once
#include <algorithm>

#include "common.cuh"

// One sweep unit = up to nv trajectories that share the impact parameter b (hence the same matrices).
struct SweepUnit { int group; int n; int traj[4]; };
constexpr int SWEEP_NV = 4;

struct Sweep1Args {          // one-centre: S = I, H = D^T (eq. (5))
    const SweepUnit *units;
    const double *D;         // [group][n_idx][N][ldD] real D^T without time phase, ldD = N rounded up to even
    const int *st_rad; const double *eps;   // per state radial index, per radial energy
    const double *v;         // [n_traj]
    double *C;               // [n_traj][N] complex amplitudes (in/out)
    double *drift;           // [n_traj] running max |sum|c|^2 - 1| (in/out) or nullptr
    int N, n_rad, n_idx;     // n_idx = half-step positions in this window (2 * steps + 1)
    int ldD, nv, rows_per_chunk, ring_stages;   // row stride of D; trajectories per unit (smem layout); rows of D per ring chunk; ring depth
    int steps;               // RK4 steps in this window
    const double *zh;        // [n_idx] z of the window's half-step positions (zh[2 s] step start, zh[2 s + 1] midpoint)
    const double *hs;        // [steps] step sizes h_s = z_{s+1} - z_s (Algorithm 1: z_mid = z + h/2, z_new = z + h)
};
inline int wp_sweep1_ld(int N) { return (N + 1) & ~1; }     // even row stride: rows are whole 16-byte units (TMA bulk copies)
void wp_sweep1_plan(int N, int n_rad, int *nv, int *rows_per_chunk, int *stages);
int wp_sweep_one_centre(wpccc_basis *B, int n_units, const Sweep1Args &a, cudaStream_t s);

struct Sweep2Args {          // two-centre: S = [[I, K^H], [K, I]], H full (eq. (1)-(4))
    const double *H;         // [traj][n_idx][N][N] complex H0^T (the TRANSPOSE: row c holds column c of H0), no time phase
    const double *K;         // [traj][n_idx][NP][NT] complex S_PT, no time phase
    const double *KT;        // [traj][n_idx][NT][NP] complex S_PT^T
    const double *Ainv;      // [traj][n_idx][NP][NP] complex (I - K K^H)^{-1}, row-major
    const int *st_rad_T, *st_rad_P; const double *eps_T, *eps_P;
    const double *v;
    double *C; double *drift;
    int NT, NP, n_idx, steps;
    const double *zh, *hs;   // as in Sweep1Args
    int solve;               // 0: Ainv holds (I - K K^H)^{-1};  1: Ainv holds the blocked Cholesky factor (wp_factor)
    const int *flags;        // [traj][n_idx] != 0: the overlap factorisation failed at this position (or nullptr)
    int *traj_status;        // [traj] 0, or 1 + global half-step index of the first failed position on the trajectory's way
    long long i0;            // global half-step index of the window's first position
};
int wp_sweep_two_centre(wpccc_basis *B, int n_traj, const Sweep2Args &a, cudaStream_t s);

// a7, solve route 0: blocked Cholesky factor A = I - K K^H = L L^H in blocks of CHOL_NB rows, stored per position in two
// packed copies so that each triangular solve of an RK4 stage streams contiguous chunks (one TMA bulk copy each):
//   Lr  block row j    : rows of block j, columns 0 .. 32 j + nb_j  ([nb_j][len_j], len_j = 32 j + nb_j): L to the left of the
//                        diagonal block, then the INVERSE of the diagonal block, Linv_jj (lower triangular);
//   Lc  block column j : rows 32 j .. n of the columns of block j ([n - 32 j][nb_j]): Linv_jj, then L below it.
// Forward solve  L w = y   : w_j = Linv_jj (y_j - sum_{i<j} L_ji w_i)          (block rows of Lr, j ascending)
// Backward solve L^H x = w : x_j = Linv_jj^H (w_j - sum_{i>j} L_ij^H x_i)      (block columns of Lc, j descending)
constexpr int CHOL_NB = 32;
struct CholLayout {
    int n, nblk;
    __host__ __device__ explicit CholLayout(int n_) : n(n_), nblk((n_ + CHOL_NB - 1) / CHOL_NB) {}
    __host__ __device__ int nb(int j) const { return min(CHOL_NB, n - CHOL_NB * j); }
    __host__ __device__ int len(int j) const { return CHOL_NB * j + nb(j); }
    __host__ __device__ size_t off_r(int j) const { return (size_t)CHOL_NB * CHOL_NB * ((size_t)j * (j + 1) / 2); }           // complex elements
    __host__ __device__ size_t size_r() const { return off_r(nblk - 1) + (size_t)nb(nblk - 1) * n; }
    __host__ __device__ size_t off_c(int j) const { return size_r() + (size_t)CHOL_NB * ((size_t)n * j - (size_t)CHOL_NB * j * (j - 1) / 2); }
    __host__ __device__ size_t size() const { return off_c(nblk - 1) + (size_t)nb(nblk - 1) * nb(nblk - 1); }                // per position
};
// complex elements per position of the factor buffer of wp_factor (either route)
__host__ __device__ inline size_t wp_factor_elems(int NP) { const size_t a = (size_t)NP * NP, b = CholLayout(NP).size(); return a > b ? a : b; }
// scratch of the Cholesky route: the Schur complement of every position of a launch, n x n complex each
size_t wp_factor_scratch_bytes(const wpccc_basis *B, int n_pos);
