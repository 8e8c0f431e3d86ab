// a0 staging: wpccc_basis_bytes / wpccc_setup_basis / wpccc_free_basis and the small query functions.
// Host side: angular coefficient tables of eq. (6) (factorials restored, A3),
// entry lists, Gauss-Legendre rules.  Device side: pair-product matrix for eq. (7), transposed radial tables
// for the five-point interpolation, r^lambda tables.
#include <cmath>
#include <cstdarg>
#include <cstring>

#include "common.cuh"

static thread_local char g_err[512] = "";
void wp_set_error(const char *fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap);
}
extern "C" const char *wpccc_last_error(void) { return g_err; }
extern "C" const char *wpccc_version(void) { return "wpccc-b200 0.1 (sm_100a)"; }

namespace {

long double lfact(int n) { long double f = 1.0L; for (int i = 2; i <= n; ++i) f *= i; return f; }

// <j1 m1; j2 m2 | J M>, integer momenta (Racah's formula, long double accumulation).
double clebsch(int j1, int m1, int j2, int m2, int J, int M) {
    if (m1 + m2 != M || J < std::abs(j1 - j2) || J > j1 + j2) return 0.0;
    if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(M) > J) return 0.0;
    long double pre = (2 * J + 1) * lfact(J + j1 - j2) * lfact(J - j1 + j2) * lfact(j1 + j2 - J) / lfact(j1 + j2 + J + 1);
    pre *= lfact(J + M) * lfact(J - M) * lfact(j1 - m1) * lfact(j1 + m1) * lfact(j2 - m2) * lfact(j2 + m2);
    long double sum = 0.0L;
    for (int k = 0; k <= j1 + j2 - J; ++k) {
        int d[6] = {k, j1 + j2 - J - k, j1 - m1 - k, j2 + m2 - k, J - j2 + m1 + k, J - j1 - m2 + k};
        bool ok = true; long double den = 1.0L;
        for (int x : d) { if (x < 0) { ok = false; break; } den *= lfact(x); }
        if (ok) sum += ((k & 1) ? -1.0L : 1.0L) / den;
    }
    return (double)(sqrtl(pre) * sum);
}

// G^lambda_{(l'm'),(lm)} = sqrt[(2l+1)(lambda-mu)!/((2l'+1)(lambda+mu)!)] <lambda 0; l 0|l' 0> <lambda mu; l m|l' m'>
double direct_G(int lp, int mp, int l, int m, int lam) {
    int mu = mp - m;
    if (std::abs(mu) > lam || lam < std::abs(lp - l) || lam > lp + l || ((lp + l + lam) & 1)) return 0.0;
    long double pref = sqrtl((long double)(2 * l + 1) * lfact(lam - mu) / ((long double)(2 * lp + 1) * lfact(lam + mu)));
    return (double)pref * clebsch(lam, 0, l, 0, lp, 0) * clebsch(lam, mu, l, m, lp, mp);
}

// n-point Gauss-Legendre rule on [-1, 1] by Newton iteration on P_n (long double), nodes ascending.
void gauss_legendre(int n, double *x, double *w) {
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < (n + 1) / 2; ++i) {
        long double z = cosl(pi * (i + 0.75L) / (n + 0.5L)), pp = 1.0L;
        for (int it = 0; it < 100; ++it) {
            long double p1 = 1.0L, p2 = 0.0L;
            for (int j = 1; j <= n; ++j) { long double p3 = p2; p2 = p1; p1 = ((2 * j - 1) * z * p2 - (j - 1) * p3) / j; }
            pp = n * (z * p1 - p2) / (z * z - 1.0L);
            long double dz = p1 / pp; z -= dz;
            if (fabsl(dz) < 1e-19L) break;
        }
        // recompute derivative at the converged node
        long double p1 = 1.0L, p2 = 0.0L;
        for (int j = 1; j <= n; ++j) { long double p3 = p2; p2 = p1; p1 = ((2 * j - 1) * z * p2 - (j - 1) * p3) / j; }
        pp = n * (z * p1 - p2) / (z * z - 1.0L);
        long double ww = 2.0L / ((1.0L - z * z) * pp * pp);
        x[i] = (double)(-z); x[n - 1 - i] = (double)z;
        w[i] = (double)ww; w[n - 1 - i] = (double)ww;
    }
    if (n & 1) x[n / 2] = 0.0;
}

// n-point Gauss-Laguerre rule: nodes x_i ascending and SCALED weights w_i e^{x_i} (the plain weights underflow).
// Nodes = eigenvalues of the Jacobi matrix (diagonal 2k + 1, off-diagonal k), isolated by Sturm-sequence bisection and
// polished by Newton's method on L_n; w_i e^{x_i} = x_i / ((n + 1) s_{n+1}(x_i))^2 with s_k = L_k(x) e^{-x/2}
// ((k + 1) s_{k+1} = (2k + 1 - x) s_k - k s_{k-1}).  Long double throughout.
void gauss_laguerre_scaled(int n, double *x, double *wx) {
    auto count_below = [&](long double t) {           // eigenvalues of the Jacobi matrix smaller than t
        int cnt = 0; long double q = 1.0L;
        for (int k = 0; k < n; ++k) {
            q = (2 * k + 1) - t - (k > 0 ? (long double)k * k / q : 0.0L);
            if (q == 0.0L) q = 1e-300L;
            if (q < 0.0L) ++cnt;
        }
        return cnt;
    };
    for (int i = 0; i < n; ++i) {
        long double lo = 0.0L, hi = 4.0L * n + 3.0L;
        for (int it = 0; it < 200 && hi - lo > 1e-12L * hi; ++it) { const long double mid = 0.5L * (lo + hi); if (count_below(mid) > i) hi = mid; else lo = mid; }
        long double z = 0.5L * (lo + hi);
        for (int it = 0; it < 8; ++it) {                // Newton on L_n: x L_n' = n (L_n - L_{n-1})
            long double s0 = expl(-0.5L * z), s1 = (1.0L - z) * s0;          // s_0, s_1
            for (int k = 1; k < n; ++k) { const long double s2 = ((2 * k + 1 - z) * s1 - k * s0) / (k + 1); s0 = s1; s1 = s2; }
            const long double ln = (n == 1) ? s1 : s1, lnm1 = s0;
            const long double dz = z * ln / (n * (ln - lnm1));
            z -= dz;
            if (fabsl(dz) < 1e-18L * fabsl(z)) break;
        }
        long double s0 = expl(-0.5L * z), s1 = (1.0L - z) * s0;
        for (int k = 1; k <= n; ++k) { const long double s2 = ((2 * k + 1 - z) * s1 - k * s0) / (k + 1); s0 = s1; s1 = s2; }
        x[i] = (double)z; wx[i] = (double)(z / (((long double)(n + 1) * s1) * ((long double)(n + 1) * s1)));
    }
}

struct Bump {
    char *base; size_t off = 0;
    explicit Bump(char *b) : base(b) {}
    template <class T> T *take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

int fill_centre_host(CentreTab &C, const wpccc_centre &in, int lambda_max) {
    C.Z = in.Z; C.n_rad = in.n_rad;
    C.l.assign(in.l, in.l + in.n_rad);
    C.eps.assign(in.eps, in.eps + in.n_rad);
    C.kind.assign(in.n_rad, 0); C.nq.assign(in.n_rad, 0);
    if (in.kind) C.kind.assign(in.kind, in.kind + in.n_rad);
    if (in.nq) C.nq.assign(in.nq, in.nq + in.n_rad);
    C.l_max = 0;
    C.st_rad.clear(); C.st_l.clear(); C.st_m.clear(); C.rad_first.clear();
    for (int a = 0; a < C.n_rad; ++a) {
        int l = C.l[a];
        if (l < 0 || l > WP_MAX_L) return -1;
        C.l_max = std::max(C.l_max, l);
        C.rad_first.push_back((int)C.st_rad.size());
        for (int m = -l; m <= l; ++m) { C.st_rad.push_back(a); C.st_l.push_back(l); C.st_m.push_back(m); }
    }
    C.n_states = (int)C.st_rad.size();
    C.n_pairs = C.n_rad * (C.n_rad + 1) / 2;
    // entries grouped by lambda: (a' <= a) with |l'-l| <= lambda <= l'+l, l'+l+lambda even (eq. (6) selection rules)
    C.lam_off.assign(WP_MAX_LAMBDA + 2, 0);
    C.ent_a1.clear(); C.ent_a.clear(); C.ent_lam.clear(); C.ent_pair.clear();
    for (int lam = 0; lam <= lambda_max; ++lam) {
        C.lam_off[lam] = (int)C.ent_a.size();
        for (int a1 = 0; a1 < C.n_rad; ++a1)
            for (int a = a1; a < C.n_rad; ++a) {
                int l1 = C.l[a1], l = C.l[a];
                if (lam < std::abs(l1 - l) || lam > l1 + l || ((l1 + l + lam) & 1)) continue;
                C.ent_a1.push_back(a1); C.ent_a.push_back(a); C.ent_lam.push_back(lam);
                C.ent_pair.push_back(a1 * C.n_rad - a1 * (a1 - 1) / 2 + (a - a1));
            }
    }
    for (int lam = lambda_max + 1; lam < WP_MAX_LAMBDA + 2; ++lam) C.lam_off[lam] = (int)C.ent_a.size();
    C.E = (int)C.ent_a.size();
    // pair-major slots of the entries (direct assembly stages F in this order): pair (a' <= a), then lambda ascending
    C.pair_off.assign(C.n_pairs + 1, 0);
    for (int e = 0; e < C.E; ++e) C.pair_off[C.ent_pair[e] + 1]++;
    for (int q = 0; q < C.n_pairs; ++q) C.pair_off[q + 1] += C.pair_off[q];
    C.ent_perm.assign(C.E, 0);
    for (int e = 0; e < C.E; ++e) {
        const int l1 = C.l[C.ent_a1[e]], l = C.l[C.ent_a[e]];
        C.ent_perm[e] = C.pair_off[C.ent_pair[e]] + (C.ent_lam[e] - std::abs(l1 - l)) / 2;
    }
    C.st_pack.resize(C.n_states);
    for (int i = 0; i < C.n_states; ++i) C.st_pack[i] = C.st_rad[i] | (C.st_l[i] << 16) | (lm_index(C.st_l[i], C.st_m[i]) << 20);
    // transfer columns (a, q >= 0) grouped by q
    C.col_rad.clear(); C.col_q.clear(); C.q_off.clear();
    for (int q = 0; q <= C.l_max; ++q) {
        C.q_off.push_back((int)C.col_rad.size());
        for (int a = 0; a < C.n_rad; ++a) if (C.l[a] >= q) { C.col_rad.push_back(a); C.col_q.push_back(q); }
    }
    C.q_off.push_back((int)C.col_rad.size());
    C.nqc = (int)C.col_rad.size();
    C.nqc_pad = (C.nqc + 7) / 8 * 8;
    C.nf_pad = 2 * C.n_rad;
    return 0;
}

// Lays the arena out; with base == nullptr only computes the size.
size_t layout(wpccc_basis &B, char *base) {
    Bump bump(base);
    const int L1 = B.lambda_max + 1;
    B.d_rp = bump.take<double>((size_t)L1 * B.Kpad);
    B.d_rm = bump.take<double>((size_t)L1 * B.Kpad);
    B.d_rk = bump.take<double>(B.Kpad);
    double *rgrid = bump.take<double>(B.Nr + 1);
    if (B.d_rgrid || !base) B.d_rgrid = base ? rgrid : reinterpret_cast<double *>(1);   // kept only for non-uniform grids (flag set by the caller)
    B.d_tiles = bump.take<GemmTile>(B.tiles.size());
    B.d_ent_lam = bump.take<int>(B.E_tot);
    B.d_st_rad_glob = bump.take<int>(B.n_tot); B.d_rad_info = bump.take<int>(B.n_rad_tot); B.d_scratch = bump.take<char>(WP_SCRATCH_BYTES);
    if (B.has_quad) {
        B.d_gl_rho = bump.take<double>(2 * (size_t)B.quad.n_rho);
        B.d_gl_phi = bump.take<double>(2 * (size_t)std::max(B.quad.n_phi, 512));
        B.d_gl_zq = bump.take<double>(2 * (size_t)(B.quad.n_z / 4));
        B.d_gl_zh = bump.take<double>(2 * (size_t)B.quad.n_z);        // kind 0: n_z/2 nodes of the middle panel; kind 1: n_z nodes in tau
    }
    for (int ci = 0; ci < B.n_centres; ++ci) {
        CentreTab &C = B.c[ci];
        const int nlm = (C.l_max + 1) * (C.l_max + 1);
        C.d_PP = bump.take<double>((size_t)C.n_pairs * B.Kpad);
        C.d_ent_pair = bump.take<int>(C.E);
        C.d_ent_lookup = bump.take<int>((size_t)L1 * C.n_rad * C.n_rad);
        C.d_G = bump.take<double>((size_t)nlm * nlm * L1);
        C.d_pair_off = bump.take<int>(C.n_pairs + 1); C.d_ent_perm = bump.take<int>(C.E); C.d_st_pack = bump.take<int>(C.n_states);
        C.d_Ut = bump.take<double>((size_t)(B.Nr + 1) * C.nf_pad);
        C.d_st_rad = bump.take<int>(C.n_states); C.d_st_l = bump.take<int>(C.n_states); C.d_st_m = bump.take<int>(C.n_states);
        C.d_eps = bump.take<double>(C.n_rad); C.d_l = bump.take<int>(C.n_rad); C.d_rad_first = bump.take<int>(C.n_rad);
        C.d_col_rad = bump.take<int>(C.nqc_pad); C.d_col_q = bump.take<int>(C.nqc_pad);
    }
    return (bump.off + 255) & ~(size_t)255;
}

int describe(wpccc_basis &B, int n_centres, const wpccc_centre *centres, int Nr, int lambda_max, const wpccc_quad *quad) {
    if (n_centres < 1 || n_centres > 2 || !centres) { wp_set_error("n_centres must be 1 or 2"); return WPCCC_EINVAL; }
    if (Nr < 8) { wp_set_error("Nr must be >= 8"); return WPCCC_EINVAL; }
    if (lambda_max < 0 || lambda_max > WP_MAX_LAMBDA) { wp_set_error("lambda_max out of range 0..%d", WP_MAX_LAMBDA); return WPCCC_EINVAL; }
    if ((n_centres == 2) != (quad != nullptr)) { wp_set_error("quad must be given iff n_centres == 2"); return WPCCC_EINVAL; }
    B.n_centres = n_centres; B.Nr = Nr; B.lambda_max = lambda_max;
    B.Kpad = (Nr + 31) / 32 * 32;
    B.has_quad = quad != nullptr;
    if (quad) {
        B.quad = *quad;
        if (quad->kind == 0 && (quad->n_rho < 1 || quad->n_phi < 1 || quad->n_z < 16 || quad->n_z % 16 || quad->rho_max <= 0 || quad->z_pad <= 0 ||
            quad->phi_rule < 0 || quad->phi_rule > 1)) { wp_set_error("bad wpccc_quad (n_z must be a multiple of 16)"); return WPCCC_EINVAL; }
        if (quad->kind == 1 && (quad->n_rho < 1 || quad->n_rho > 128 || quad->n_z < 16 || quad->n_z % 16 || !(quad->eta_scale > 0))) {
            wp_set_error("bad spheroidal wpccc_quad (1 <= n_rho <= 128 Laguerre nodes, n_z a multiple of 16, eta_scale > 0)"); return WPCCC_EINVAL; }
        if (quad->kind < 0 || quad->kind > 1) { wp_set_error("wpccc_quad.kind must be 0 or 1"); return WPCCC_EINVAL; }
    }
    B.n_tot = 0; B.E_tot = 0; B.n_rad_tot = 0; B.tiles.clear();
    for (int ci = 0; ci < n_centres; ++ci) {
        if (centres[ci].n_rad < 1 || centres[ci].n_rad > 60000 || !centres[ci].l || !centres[ci].eps || !centres[ci].u) { wp_set_error("centre %d: missing arrays", ci); return WPCCC_EINVAL; }
        if (fill_centre_host(B.c[ci], centres[ci], lambda_max)) { wp_set_error("centre %d: l out of range 0..%d", ci, WP_MAX_L); return WPCCC_EINVAL; }
        B.n_tot += B.c[ci].n_states; B.E_tot += B.c[ci].E; B.n_rad_tot += B.c[ci].n_rad;
        for (int lam = 0; lam <= lambda_max; ++lam) {
            int cnt = B.c[ci].lam_off[lam + 1] - B.c[ci].lam_off[lam];
            for (int n0 = 0; n0 < cnt; n0 += 128) B.tiles.push_back(GemmTile{ci, lam, n0, std::min(128, cnt - n0)});
        }
    }
    return 0;
}

__global__ void k_pair_products(const double *Ut, int nf_pad, int n_rad, const double *w, int Nr, int Kpad, double *PP) {
    // PP[pair(a1,a)][k-1] = w_k u_a1(r_k) u_a(r_k), k = 1..Nr; zero for k-1 >= Nr
    const int pair = blockIdx.x;                     // pairs along x: there can be more than 65 535 of them
    int a1 = 0, rem = pair;
    while (rem >= n_rad - a1) { rem -= n_rad - a1; ++a1; }
    const int a = a1 + rem;
    for (int kk = blockIdx.y * blockDim.x + threadIdx.x; kk < Kpad; kk += gridDim.y * blockDim.x) {
        double v = 0.0;
        if (kk < Nr) { const double *row = Ut + (size_t)(kk + 1) * nf_pad; v = w[kk + 1] * row[2 * a1] * row[2 * a]; }
        PP[(size_t)pair * Kpad + kk] = v;
    }
}

template <class T> int upload(T *dst, const std::vector<T> &src, cudaStream_t s) {
    if (src.empty()) return 0;
    WP_CUDA(cudaMemcpyAsync(dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s));
    return 0;
}

}  // namespace

extern "C" size_t wpccc_basis_bytes(int n_centres, const wpccc_centre *centres, int Nr, int lambda_max, const wpccc_quad *quad) {
    wpccc_basis B;
    if (describe(B, n_centres, centres, Nr, lambda_max, quad)) return 0;
    return layout(B, nullptr) + (size_t)(Nr + 1) * sizeof(double) + 256;   // + scratch for the weights
}

static int setup_impl(wpccc_basis **out, int n_centres, const wpccc_centre *centres, double Z_proj, int Nr, double h, const double *rgrid,
                      const double *w, int lambda_max, const wpccc_quad *quad, void *dev_arena, size_t arena_bytes, void *stream) {
    if (!out) WP_FAIL(WPCCC_EINVAL, "out is NULL");
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) WP_FAIL(WPCCC_ECUDA, "no CUDA device (this library has no CPU fallback)");
    if (!w || (!rgrid && !(h > 0))) WP_FAIL(WPCCC_EINVAL, "w is NULL or h <= 0");
    if (rgrid) {
        if (rgrid[0] != 0.0) WP_FAIL(WPCCC_EINVAL, "r[0] must be 0");
        for (int k = 0; k < Nr; ++k) if (!(rgrid[k + 1] > rgrid[k])) WP_FAIL(WPCCC_EINVAL, "radial grid must be strictly increasing (index %d)", k);
        h = rgrid[Nr] / Nr;                            // only a scale (initial guesses of index searches)
    }
    if (!dev_arena || ((uintptr_t)dev_arena & 255)) WP_FAIL(WPCCC_EINVAL, "dev_arena must be a 256-byte aligned device pointer");
    wpccc_basis *B = new wpccc_basis;
    int rc = describe(*B, n_centres, centres, Nr, lambda_max, quad);
    if (rc) { delete B; return rc; }
    if (n_centres == 2 && Z_proj != centres[1].Z) { delete B; WP_FAIL(WPCCC_EINVAL, "Z_proj must equal centres[1].Z with two centres"); }
    B->h = h; B->Z_proj = Z_proj;
    B->d_rgrid = rgrid ? reinterpret_cast<double *>(1) : nullptr;     // layout() turns the flag into the arena pointer
    const size_t need = layout(*B, (char *)dev_arena);
    const size_t w_off = need;
    if (arena_bytes < need + (size_t)(Nr + 1) * sizeof(double)) { delete B; WP_FAIL(WPCCC_ENOMEM, "arena too small: need %zu bytes", need + (size_t)(Nr + 1) * 8); }
    B->arena = (char *)dev_arena; B->arena_bytes = arena_bytes;
    cudaStream_t s = (cudaStream_t)stream;
    double *d_w = reinterpret_cast<double *>((char *)dev_arena + w_off);

    // r^lambda tables (k = 1..Nr at index k-1; padding rows are zero so that V = 0 there)
    const int L1 = lambda_max + 1;
    std::vector<double> rp((size_t)L1 * B->Kpad, 0.0), rm((size_t)L1 * B->Kpad, 0.0), rk(B->Kpad, 0.0);
    for (int kk = 0; kk < Nr; ++kk) {
        const double r = rgrid ? rgrid[kk + 1] : h * (double)(kk + 1);
        rk[kk] = r;
        double p = 1.0;
        for (int lam = 0; lam < L1; ++lam) { rp[(size_t)lam * B->Kpad + kk] = p; rm[(size_t)lam * B->Kpad + kk] = 1.0 / (p * r); p *= r; }
    }
    std::vector<cudaError_t> errs;
    auto chk = [&](int r_) { if (r_ && !rc) rc = r_; };
    chk(upload(B->d_rp, rp, s)); chk(upload(B->d_rm, rm, s)); chk(upload(B->d_rk, rk, s));
    if (rgrid && !rc && cudaMemcpyAsync(B->d_rgrid, rgrid, (size_t)(Nr + 1) * sizeof(double), cudaMemcpyHostToDevice, s) != cudaSuccess) rc = WPCCC_ECUDA;
    chk(upload(B->d_tiles, B->tiles, s));
    std::vector<int> all_lam;
    for (int ci = 0; ci < n_centres; ++ci) all_lam.insert(all_lam.end(), B->c[ci].ent_lam.begin(), B->c[ci].ent_lam.end());
    chk(upload(B->d_ent_lam, all_lam, s));
    std::vector<int> st_rad_glob, rad_info;
    for (int ci = 0, off = 0; ci < n_centres; off += B->c[ci].n_rad, ++ci) {
        for (int j = 0; j < B->c[ci].n_states; ++j) st_rad_glob.push_back(off + B->c[ci].st_rad[j]);
        for (int a = 0; a < B->c[ci].n_rad; ++a) rad_info.push_back(2 * ci + (B->c[ci].kind[a] != 0));
    }
    chk(upload(B->d_st_rad_glob, st_rad_glob, s)); chk(upload(B->d_rad_info, rad_info, s));
    if (!rc && cudaMemcpyAsync(d_w, w, (size_t)(Nr + 1) * sizeof(double), cudaMemcpyHostToDevice, s) != cudaSuccess) rc = WPCCC_ECUDA;
    std::vector<std::vector<double>> keep_d; std::vector<std::vector<int>> keep_i;   // host staging must outlive the async copies
    if (!rc && B->has_quad) {
        auto rule = [&](int n, double *dst) {
            keep_d.emplace_back(2 * (size_t)n);
            gauss_legendre(n, keep_d.back().data(), keep_d.back().data() + n);
            chk(upload(dst, keep_d.back(), s));
        };
        if (B->quad.kind == 1) {
            keep_d.emplace_back(2 * (size_t)B->quad.n_rho);
            gauss_laguerre_scaled(B->quad.n_rho, keep_d.back().data(), keep_d.back().data() + B->quad.n_rho);
            chk(upload(B->d_gl_rho, keep_d.back(), s));
            rule(B->quad.n_z, B->d_gl_zh);
        } else {
            rule(B->quad.n_rho, B->d_gl_rho);
            if (B->quad.phi_rule == 0) rule(B->quad.n_phi, B->d_gl_phi);
            rule(B->quad.n_z / 4, B->d_gl_zq);
            rule(B->quad.n_z / 2, B->d_gl_zh);
        }
    }
    for (int ci = 0; ci < n_centres && !rc; ++ci) {
        CentreTab &C = B->c[ci];
        const int nlm = (C.l_max + 1) * (C.l_max + 1);
        keep_d.emplace_back((size_t)nlm * nlm * L1, 0.0);
        std::vector<double> &G = keep_d.back();
        for (int lp = 0; lp <= C.l_max; ++lp) for (int mp = -lp; mp <= lp; ++mp)
            for (int l = 0; l <= C.l_max; ++l) for (int m = -l; m <= l; ++m)
                for (int lam = 0; lam < L1; ++lam)
                    G[((size_t)lm_index(lp, mp) * nlm + lm_index(l, m)) * L1 + lam] = direct_G(lp, mp, l, m, lam);
        chk(upload(C.d_G, G, s));
        keep_i.emplace_back((size_t)L1 * C.n_rad * C.n_rad, -1);
        std::vector<int> &look = keep_i.back();
        for (int e = 0; e < C.E; ++e) look[((size_t)C.ent_lam[e] * C.n_rad + C.ent_a1[e]) * C.n_rad + C.ent_a[e]] = e;
        chk(upload(C.d_ent_lookup, look, s));
        chk(upload(C.d_ent_pair, C.ent_pair, s));
        chk(upload(C.d_pair_off, C.pair_off, s)); chk(upload(C.d_ent_perm, C.ent_perm, s)); chk(upload(C.d_st_pack, C.st_pack, s));
        chk(upload(C.d_st_rad, C.st_rad, s)); chk(upload(C.d_st_l, C.st_l, s)); chk(upload(C.d_st_m, C.st_m, s));
        chk(upload(C.d_eps, C.eps, s)); chk(upload(C.d_l, C.l, s)); chk(upload(C.d_rad_first, C.rad_first, s));
        keep_i.emplace_back(C.col_rad); keep_i.back().resize(C.nqc_pad, -1); chk(upload(C.d_col_rad, keep_i.back(), s));
        keep_i.emplace_back(C.col_q); keep_i.back().resize(C.nqc_pad, 0); chk(upload(C.d_col_q, keep_i.back(), s));
        // transposed radial table: row k = [(u_0, g_0), (u_1, g_1), ...] at r_k
        keep_d.emplace_back((size_t)(Nr + 1) * C.nf_pad, 0.0);
        std::vector<double> &Ut = keep_d.back();
        for (int a = 0; a < C.n_rad; ++a)
            for (int k = 0; k <= Nr; ++k) {
                Ut[(size_t)k * C.nf_pad + 2 * a] = centres[ci].u[(size_t)a * (Nr + 1) + k];
                Ut[(size_t)k * C.nf_pad + 2 * a + 1] = centres[ci].g ? centres[ci].g[(size_t)a * (Nr + 1) + k] : 0.0;
            }
        chk(upload(C.d_Ut, Ut, s));
        if (!rc) {
            dim3 grid(C.n_pairs, std::min((B->Kpad + 255) / 256, 64));
            k_pair_products<<<grid, 256, 0, s>>>(C.d_Ut, C.nf_pad, C.n_rad, d_w, Nr, B->Kpad, C.d_PP);
            if (cudaGetLastError() != cudaSuccess) { wp_set_error("k_pair_products launch failed"); rc = WPCCC_ECUDA; }
        }
    }
    if (!rc && cudaStreamSynchronize(s) != cudaSuccess) { wp_set_error("setup: stream synchronize failed"); rc = WPCCC_ECUDA; }
    if (!rc) {
        int pr_least = 0, pr_greatest = 0;
        cudaDeviceGetStreamPriorityRange(&pr_least, &pr_greatest);
        if (cudaStreamCreateWithPriority(&B->side, cudaStreamNonBlocking, pr_least) != cudaSuccess ||
            cudaStreamCreateWithPriority(&B->hi, cudaStreamNonBlocking, pr_greatest) != cudaSuccess ||
            cudaEventCreateWithFlags(&B->ev_join2, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&B->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&B->ev_join, cudaEventDisableTiming) != cudaSuccess) { wp_set_error("stream/event creation failed"); rc = WPCCC_ECUDA; }
    }
    if (rc) { delete B; return rc; }
    *out = B;
    return 0;
}

extern "C" int wpccc_setup_basis(wpccc_basis **out, int n_centres, const wpccc_centre *centres, double Z_proj, int Nr, double h,
                                 const double *w, int lambda_max, const wpccc_quad *quad, void *dev_arena, size_t arena_bytes,
                                 void *stream) {
    return setup_impl(out, n_centres, centres, Z_proj, Nr, h, nullptr, w, lambda_max, quad, dev_arena, arena_bytes, stream);
}

extern "C" int wpccc_setup_basis_grid(wpccc_basis **out, int n_centres, const wpccc_centre *centres, double Z_proj, int Nr, const double *r,
                                      const double *w, int lambda_max, const wpccc_quad *quad, void *dev_arena, size_t arena_bytes,
                                      void *stream) {
    if (!r) WP_FAIL(WPCCC_EINVAL, "r is NULL");
    return setup_impl(out, n_centres, centres, Z_proj, Nr, 0.0, r, w, lambda_max, quad, dev_arena, arena_bytes, stream);
}

extern "C" void wpccc_free_basis(wpccc_basis *B) {
    if (!B) return;
    for (auto e : B->ev_pool) cudaEventDestroy(e);
    if (B->ev_fork) cudaEventDestroy(B->ev_fork);
    if (B->ev_join) cudaEventDestroy(B->ev_join);
    if (B->ev_join2) cudaEventDestroy(B->ev_join2);
    if (B->side) cudaStreamDestroy(B->side);
    if (B->hi) cudaStreamDestroy(B->hi);
    delete B;
}

extern "C" int wpccc_n_states(const wpccc_basis *B) { return B ? B->n_tot : WPCCC_EINVAL; }
extern "C" int wpccc_n_states_centre(const wpccc_basis *B, int c) { return (B && c >= 0 && c < B->n_centres) ? B->c[c].n_states : WPCCC_EINVAL; }
extern "C" int wpccc_n_rad_centre(const wpccc_basis *B, int c) { return (B && c >= 0 && c < B->n_centres) ? B->c[c].n_rad : WPCCC_EINVAL; }
extern "C" int wpccc_n_radial_entries(const wpccc_basis *B, int c) { return (B && c >= 0 && c < B->n_centres) ? B->c[c].E : WPCCC_EINVAL; }
extern "C" int wpccc_radial_entry(const wpccc_basis *B, int c, int e, int *a1, int *a, int *lam) {
    if (!B || c < 0 || c >= B->n_centres || e < 0 || e >= B->c[c].E) WP_FAIL(WPCCC_EINVAL, "bad centre/entry index");
    if (a1) *a1 = B->c[c].ent_a1[e];
    if (a) *a = B->c[c].ent_a[e];
    if (lam) *lam = B->c[c].ent_lam[e];
    return 0;
}

// ---- timing spans ----
static cudaEvent_t take_event(wpccc_basis *B) {
    if (B->ev_used == B->ev_pool.size()) { cudaEvent_t e; cudaEventCreate(&e); B->ev_pool.push_back(e); }
    return B->ev_pool[B->ev_used++];
}
void wp_timing_reset(wpccc_basis *B) {
    B->spans.clear(); B->ev_used = 0;
    for (int k = 0; k < WP_NFAM; ++k) { B->launches[k] = 0; B->groups[k] = 0; B->units[k] = 0; }
}
// Spans are sampled: families launched once per chunk of positions (thousands of launches per call) record an
// event pair on every 8th launch group only; the family total is the sampled mean times the number of groups.
static const int k_sample_every[WP_NFAM] = {1, 1, 8, 8, 1, 1, 1, 1};
void wp_span_begin(wpccc_basis *B, int fam, cudaStream_t s) {
    B->cur_fam = fam;
    B->cur_sampled = (B->groups[fam]++ % k_sample_every[fam]) == 0 && B->opt.timing;
    if (!B->cur_sampled) return;
    wpccc_basis::Span sp; sp.fam = fam; sp.a = take_event(B); sp.b = take_event(B);
    cudaEventRecord(sp.a, s);
    B->spans.push_back(sp);
}
void wp_span_end(wpccc_basis *B, cudaStream_t s, int n_launches) {
    B->launches[B->cur_fam] += n_launches;
    if (!B->cur_sampled) return;
    cudaEventRecord(B->spans.back().b, s);
}
extern "C" int wpccc_last_timing(const wpccc_basis *Bc, double *ms, long long *launches) {
    if (!Bc) return WPCCC_EINVAL;
    wpccc_basis *B = const_cast<wpccc_basis *>(Bc);
    cudaDeviceSynchronize();
    long long sampled[WP_NFAM] = {0};
    for (int k = 0; k < WP_NFAM; ++k) B->last_ms[k] = 0.0;
    for (auto &sp : B->spans) { float t = 0.f; if (cudaEventElapsedTime(&t, sp.a, sp.b) == cudaSuccess) { B->last_ms[sp.fam] += t; ++sampled[sp.fam]; } }
    for (int k = 0; k < WP_NFAM; ++k) {
        if (sampled[k] > 0) B->last_ms[k] *= (double)B->groups[k] / (double)sampled[k];
        if (ms) ms[k] = B->last_ms[k];
        if (launches) launches[k] = B->launches[k];
    }
    return WP_NFAM;
}
extern "C" int wpccc_last_units(const wpccc_basis *B, long long *units) {
    if (!B || !units) return WPCCC_EINVAL;
    for (int k = 0; k < WP_NFAM; ++k) units[k] = B->units[k];
    return WP_NFAM;
}
