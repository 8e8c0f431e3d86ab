// a8: RK4 sweep kernels (Algorithm 1) -- declarations shared by api.cu and sweep.cu.
#pragma once
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
    long long i0;            // global half-step index of the window's first position
    double z_min, h;         // z_i = z_min + 0.5 * i * h
};
inline int wp_sweep1_ld(int N) { return (N + 1) & ~1; }     // even row stride: rows are whole 16-byte units (TMA bulk copies)
void wp_sweep1_plan(int N, int n_rad, int *nv, int *rows_per_chunk, int *stages);
int wp_sweep_one_centre(wpccc_basis *B, int n_units, const Sweep1Args &a, cudaStream_t s);

struct Sweep2Args {          // two-centre: S = [[I, K^H], [K, I]], H full (eq. (1)-(4))
    const double *H;         // [traj][n_idx][N][N] complex, no time phase
    const double *K;         // [traj][n_idx][NP][NT] complex S_PT, no time phase
    const double *Ainv;      // [traj][n_idx][NP][NP] complex (I - K K^H)^{-1}, row-major
    const int *st_rad_T, *st_rad_P; const double *eps_T, *eps_P;
    const double *v;
    double *C; double *drift;
    int NT, NP, n_idx, steps;
    long long i0;
    double z_min, h;
};
int wp_sweep_two_centre(wpccc_basis *B, int n_traj, const Sweep2Args &a, cudaStream_t s);
