// Host-side setup of a handle (DESIGN.md step a0): shell normalisation (R11), primitive-pair tables,
// Schwarz bounds (R14, computed on the device), class/bound sorting, a-lists and work lists, one-electron
// integrals (overlap for callers, dipoles for eq. 19), Boys table.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <numeric>
#include "common.cuh"

namespace rttda {

// ---------------------------------------------------------------------------------------------- Boys table
// Rows {F_{L+k}(T0)/k!, k = 0..7; exp(-T0); 0} at T0 = j/8 (eri_eval.cuh boys_near<L>): series for F_{L+7} (T0 <= BOYS_TMAX + 1/8),
// downward recursion for the lower orders, all in long double.
void boys_table_host(int L, std::vector<double>& tab)
{
    tab.assign((size_t)BOYS_NROW * BOYS_ROW, 0.0);
    const int n = L + 7;
    const long double fact[8] = {1, 1, 2, 6, 24, 120, 720, 5040};
    for (int j = 0; j < BOYS_NROW; ++j) {
        const long double T = (long double)j / 8.0L;
        long double term = 1.0L / (2 * n + 1), sum = term;
        for (int k = 1; k < 4000; ++k) {
            term *= 2.0L * T / (2 * n + 2 * k + 1);
            sum += term;
            if (term < 1e-21L * sum) break;
        }
        const long double emt = expl(-T);
        long double f = emt * sum;                       // F_{L+7}(T0)
        double* row = &tab[(size_t)j * BOYS_ROW];
        row[7] = (double)(f / fact[7]);
        for (int m = n; m > L; --m) {                    // F_{m-1} = (2 T F_m + e^-T) / (2m - 1)
            f = (2.0L * T * f + emt) / (2 * m - 1);
            row[m - 1 - L] = (double)(f / fact[m - 1 - L]);
        }
        row[8] = (double)emt;
    }
}

// ---------------------------------------------------------------------------------------------- basis
struct HostBasis {
    int nshells = 0, nao = 0;
    std::vector<int> l, np, np_true, off, ao, center;   // np: primitives stored (2 is padded to 3), np_true: as given
    std::vector<double> ex, cf;          // cf: final coefficient of the bare primitive
    std::vector<double> xyz;             // [ncenters][3]
};

static int load_basis(const rttda_basis_t* b, HostBasis& H)
{
    RT_CHECK(b && b->centers && b->shells && b->exps && b->coefs, "basis: NULL pointer");
    RT_CHECK(b->nshells > 0 && b->ncenters > 0, "basis: empty");
    H.nshells = b->nshells;
    H.xyz.assign(b->centers, b->centers + 3 * (size_t)b->ncenters);
    int ao = 0;
    for (int s = 0; s < b->nshells; ++s) {
        const rttda_shell_t& sh = b->shells[s];
        RT_CHECK(sh.l >= 0 && sh.l <= 2, "basis: only s, p and (Cartesian) d shells are supported");
        RT_CHECK(sh.nprim >= 1 && sh.nprim <= RTTDA_MAX_NPRIM, "basis: nprim out of range");
        RT_CHECK(sh.center >= 0 && sh.center < b->ncenters, "basis: bad centre index");
        // Contraction depths 1 and 3 have their own kernel instantiations; a 2-primitive shell is carried as a
        // 3-primitive shell whose third primitive has coefficient zero (same integrals, some idle arithmetic).
        const int np_store = sh.nprim == 2 ? 3 : sh.nprim;
        H.l.push_back(sh.l); H.np.push_back(np_store); H.np_true.push_back(sh.nprim); H.off.push_back((int)H.ex.size());
        H.center.push_back(sh.center); H.ao.push_back(ao);
        ao += ncart(sh.l);
        // Primitives are taken in order of ascending exponent: the contraction sums do not depend on the order, but
        // with every shell sorted the same way a primitive-pair index means "diffuse x diffuse" ... "tight x tight"
        // for all kets of a warp alike, which makes the near-field / far-field Boys branch of the evaluation kernels
        // (eri_eval.cuh) far more uniform across the lanes.
        std::vector<int> order(sh.nprim);
        std::iota(order.begin(), order.end(), 0);
        std::sort(order.begin(), order.end(), [&](int x, int y) { return b->exps[sh.prim_off + x] < b->exps[sh.prim_off + y]; });
        // coefficient on the normalised primitive -> coefficient on the bare primitive
        std::vector<double> c(sh.nprim);
        for (int k = 0; k < sh.nprim; ++k) {
            const double a = b->exps[sh.prim_off + order[k]];
            RT_CHECK(a > 0.0, "basis: non-positive exponent");
            double nrm = std::pow(2.0 * a / M_PI, 0.75);
            if (sh.l == 1) nrm *= 2.0 * std::sqrt(a);
            if (sh.l == 2) nrm *= 4.0 * a / std::sqrt(3.0);          // the xx component; xy, xz, yz carry sqrt(3) more (R11)
            c[k] = b->coefs[sh.prim_off + order[k]] * nrm;
            H.ex.push_back(a);
        }
        // self overlap of the contracted function: s: sum c c (pi/p)^1.5 ; p: ... / (2p) ; d (xx): ... * 3 / (4 p^2)
        double self = 0.0;
        for (int k = 0; k < sh.nprim; ++k)
            for (int m = 0; m < sh.nprim; ++m) {
                const double p = H.ex[H.off.back() + k] + H.ex[H.off.back() + m];   // sorted order, as c[]
                double t = c[k] * c[m] * std::pow(M_PI / p, 1.5);
                if (sh.l == 1) t /= 2.0 * p;
                if (sh.l == 2) t *= 0.75 / (p * p);
                self += t;
            }
        RT_CHECK(self > 0.0, "basis: contracted function has zero norm");
        for (int k = 0; k < sh.nprim; ++k) H.cf.push_back(c[k] / std::sqrt(self));
        if (np_store != sh.nprim) { H.ex.push_back(H.ex.back()); H.cf.push_back(0.0); }
    }
    H.nao = ao;
    return RTTDA_OK;
}

// One-electron block of a shell pair: S[na*nb] and D[3][na*nb] (origin 0), from the 1-D Hermite coefficients
// E_0 (overlap) and E_1 + P E_0 (first moment) of every primitive pair; Gaussian-product factor in `base`.
static void pair_1e(const HostBasis& H, int sa, int sb, double* S, double* D)
{
    const int la = H.l[sa], lb = H.l[sb], na = ncart(la), nb = ncart(lb);
    const double* A = &H.xyz[3 * H.center[sa]];
    const double* B = &H.xyz[3 * H.center[sb]];
    std::fill(S, S + na * nb, 0.0);
    std::fill(D, D + 3 * na * nb, 0.0);
    const double ab2 = (A[0] - B[0]) * (A[0] - B[0]) + (A[1] - B[1]) * (A[1] - B[1]) + (A[2] - B[2]) * (A[2] - B[2]);
    auto powers = [](int l, int c, int* pw) {              // s; x y z; xx xy xz yy yz zz
        pw[0] = pw[1] = pw[2] = 0;
        if (l == 1) pw[c] = 1;
        if (l == 2) { const int f = c < 3 ? 0 : (c < 5 ? 1 : 2), g = c < 3 ? c : (c < 5 ? c - 2 : 2); pw[f] += 1; pw[g] += 1; }
    };
    auto cnorm = [](int l, int c) { return (l == 2 && (c == 1 || c == 2 || c == 4)) ? std::sqrt(3.0) : 1.0; };
    for (int ka = 0; ka < H.np[sa]; ++ka)
        for (int kb = 0; kb < H.np[sb]; ++kb) {
            const double a = H.ex[H.off[sa] + ka], b = H.ex[H.off[sb] + kb], p = a + b;
            const double base = H.cf[H.off[sa] + ka] * H.cf[H.off[sb] + kb] * std::pow(M_PI / p, 1.5) *
                                std::exp(-a * b / p * ab2);
            double P[3], E[3][3][3][6];                     // [axis][i][j][t], t <= i + j (+1 slack)
            for (int x = 0; x < 3; ++x) {
                P[x] = (a * A[x] + b * B[x]) / p;
                const double xa = P[x] - A[x], xb = P[x] - B[x], h = 0.5 / p;
                for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int t = 0; t < 6; ++t) E[x][i][j][t] = 0.0;
                E[x][0][0][0] = 1.0;
                for (int i = 0; i < la; ++i)
                    for (int t = 0; t <= i + 1; ++t)
                        E[x][i + 1][0][t] = (t > 0 ? h * E[x][i][0][t - 1] : 0.0) + xa * E[x][i][0][t] + (t + 1) * E[x][i][0][t + 1];
                for (int i = 0; i <= la; ++i)
                    for (int j = 0; j < lb; ++j)
                        for (int t = 0; t <= i + j + 1; ++t)
                            E[x][i][j + 1][t] = (t > 0 ? h * E[x][i][j][t - 1] : 0.0) + xb * E[x][i][j][t] + (t + 1) * E[x][i][j][t + 1];
            }
            for (int ca = 0; ca < na; ++ca)
                for (int cb = 0; cb < nb; ++cb) {
                    int pa[3], pb[3];
                    powers(la, ca, pa); powers(lb, cb, pb);
                    const double cn = base * cnorm(la, ca) * cnorm(lb, cb);
                    const double f0 = E[0][pa[0]][pb[0]][0], f1 = E[1][pa[1]][pb[1]][0], f2 = E[2][pa[2]][pb[2]][0];
                    S[ca * nb + cb] += cn * f0 * f1 * f2;
                    const double m0 = E[0][pa[0]][pb[0]][1] + P[0] * f0, m1 = E[1][pa[1]][pb[1]][1] + P[1] * f1,
                                 m2 = E[2][pa[2]][pb[2]][1] + P[2] * f2;
                    D[0 * na * nb + ca * nb + cb] += cn * m0 * f1 * f2;
                    D[1 * na * nb + ca * nb + cb] += cn * f0 * m1 * f2;
                    D[2 * na * nb + ca * nb + cb] += cn * f0 * f1 * m2;
                }
        }
}

static void one_electron_host(const HostBasis& H, double* S, double* D)
{
    const size_t N = H.nao;
    for (int sa = 0; sa < H.nshells; ++sa)
        for (int sb = 0; sb < H.nshells; ++sb) {
            double s[36], d[108];
            pair_1e(H, sa, sb, s, d);
            const int na = ncart(H.l[sa]), nb = ncart(H.l[sb]);
            for (int ca = 0; ca < na; ++ca)
                for (int cb = 0; cb < nb; ++cb) {
                    const size_t idx = (size_t)(H.ao[sa] + ca) * N + H.ao[sb] + cb;
                    if (S) S[idx] = s[ca * nb + cb];
                    if (D)
                        for (int x = 0; x < 3; ++x) D[x * N * N + idx] = d[x * na * nb + ca * nb + cb];
                }
        }
}

// Primitive-pair rows of the ordered shell pair (first, second).
static void prim_rows(const HostBasis& H, int s1, int s2, std::vector<double>& rows)
{
    const double* A = &H.xyz[3 * H.center[s1]];
    const double* B = &H.xyz[3 * H.center[s2]];
    const double ab2 = (A[0] - B[0]) * (A[0] - B[0]) + (A[1] - B[1]) * (A[1] - B[1]) + (A[2] - B[2]) * (A[2] - B[2]);
    const double c0 = std::sqrt(2.0) * std::pow(M_PI, 1.25);
    for (int k1 = 0; k1 < H.np[s1]; ++k1)
        for (int k2 = 0; k2 < H.np[s2]; ++k2) {
            const double a = H.ex[H.off[s1] + k1], b = H.ex[H.off[s2] + k2], p = a + b;
            double r[PRIM_STRIDE];
            r[0] = p;
            for (int x = 0; x < 3; ++x) {
                r[1 + x] = (a * A[x] + b * B[x]) / p;
                r[6 + x] = r[1 + x] - A[x];
                r[9 + x] = r[1 + x] - B[x];
            }
            r[4] = c0 / p * H.cf[H.off[s1] + k1] * H.cf[H.off[s2] + k2] * std::exp(-a * b / p * ab2);
            r[5] = 0.5 / p;
            rows.insert(rows.end(), r, r + PRIM_STRIDE);
        }
}

__global__ void shift_diag_kernel(int n, double c, double* __restrict__ A)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) A[(size_t)i * n + i] += c;
}

struct DevTmp {                   // temporary device allocation, released on scope exit (error paths included)
    void* p = nullptr;
    ~DevTmp() { if (p) cudaFree(p); }
};

struct Pair {
    int s1, s2;          // first (higher l, or larger index at equal l), second
    int pc, sub, np;     // pair class, contraction sub-class, primitive pairs (stored)
    int np_true;         // primitive pairs as given (2-primitive shells are padded), for the R14 counters
    std::vector<int> sel; // the primitive rows kept (offsets from `row`, ascending), np of them
    int row;             // first row in the per-class candidate prim table
    double Q;
    int pos;             // position in its ket class after sorting
};

template <class T>
static int upload(Handle* h, const std::vector<T>& v, const T** out)
{
    void* d = nullptr;
    const size_t bytes = std::max<size_t>(v.size(), 1) * sizeof(T);
    RT_CUDA(cudaMalloc(&d, bytes));
    h->dev_allocs.push_back(d);
    if (!v.empty()) RT_CUDA(cudaMemcpy(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
    *out = (const T*)d;
    return RTTDA_OK;
}

static int np_to_sub(int np) { return np == 1 ? 0 : (np == 3 ? 1 : (np == 6 ? 2 : 3)); }

// Flop model of one primitive quartet of total angular momentum L, bra/ket split irrelevant at this
// granularity: geometry + prefactor, Boys, R recursion, operator stages.
double flops_prim(int la, int lb, int lc, int ld)
{
    const int L = la + lb + lc + ld;
    auto nh = [](int n) { return (n + 1) * (n + 2) * (n + 3) / 6; };
    double fma = 0.0, other = 0.0;
    other += 16;                       // P-Q, |PQ|^2, p+q, rsqrt (counted as 4), alpha, prefactor
    fma += 8 + (L > 0 ? 9 + L : 0);    // Boys Taylor (+ exp Taylor + downward recursion)
    other += L + 1;                    // (-2 alpha)^n scaling
    for (int N = 1; N <= L; ++N) fma += (double)(L - N + 1) * (nh(N) - nh(N - 1)) * 1.5;
    int ord = L, blk = 1;
    const int ls[4] = {ld, lc, lb, la};
    for (int s = 0; s < 4; ++s)
        for (int k = 0; k < ls[s]; ++k) { ord -= 1; fma += 2.0 * 3 * blk * nh(ord) * 0.75; blk *= 3; }   // d: two operator stages [est.]
    return 2.0 * fma + other;
}

double flops_prim_L(int L)
{
    static const int cls[5][4] = {{0, 0, 0, 0}, {1, 0, 0, 0}, {1, 0, 1, 0}, {1, 1, 1, 0}, {1, 1, 1, 1}};
    return flops_prim(cls[L][0], cls[L][1], cls[L][2], cls[L][3]);
}

int create_impl(Handle* h, const rttda_basis_t* basis, const double* C_occ, const double* C_virt,
                const double* eps, cudaStream_t st)
{
    auto t0 = std::chrono::steady_clock::now();
    HostBasis H;
    RT_TRY(load_basis(basis, H));
    RT_CHECK(H.nao == h->nao, "nao does not match the shell table");
    h->nshells = H.nshells;
    const size_t N = h->nao;

    // ---- Boys table
    for (int L = 0; L <= 8; ++L) {
        std::vector<double> boys;
        boys_table_host(L, boys);
        const double* d = nullptr;
        RT_TRY(upload(h, boys, &d));
        h->tabs.boys[L] = reinterpret_cast<const double2*>(d);
    }

    // ---- candidate pairs and their primitive rows (canonical orientation), per pair class
    std::vector<Pair> pairs;
    std::vector<double> rows[NPAIRCLASS];
    std::vector<int> cand_np[NPAIRCLASS], cand_off[NPAIRCLASS], cand_id[NPAIRCLASS];
    long long npairs_total = 0;
    for (int i = 0; i < H.nshells; ++i)
        for (int j = 0; j <= i; ++j) {
            ++npairs_total;
            int s1 = i, s2 = j;
            if (H.l[s2] > H.l[s1]) std::swap(s1, s2);
            Pair P;
            P.s1 = s1; P.s2 = s2; P.pc = pairclass_of(H.l[s1], H.l[s2]); P.np = H.np[s1] * H.np[s2];
            P.np_true = H.np_true[s1] * H.np_true[s2];
            RT_CHECK(P.np == 1 || P.np == 3 || P.np == 9, "unsupported contraction depth");
            P.sub = np_to_sub(P.np);
            const size_t before = rows[P.pc].size();
            prim_rows(H, s1, s2, rows[P.pc]);
            double cmax = 0.0;
            for (size_t r = before; r < rows[P.pc].size(); r += PRIM_STRIDE) cmax = std::max(cmax, std::fabs(rows[P.pc][r + 4]));
            if (cmax < 1e-30) {                 // Gaussian product vanishes: contributes < 1e-30 everywhere
                rows[P.pc].resize(before);
                continue;
            }
            P.row = (int)(before / PRIM_STRIDE);
            P.Q = 0.0; P.pos = -1;
            cand_np[P.pc].push_back(P.np);
            cand_off[P.pc].push_back(P.row);
            cand_id[P.pc].push_back((int)pairs.size());
            pairs.push_back(P);
        }

    // ---- Schwarz bounds on the device
    std::vector<double> qprim[NPAIRCLASS];
    for (int pc = 0; pc < NPAIRCLASS; ++pc) {
        const int n = (int)cand_np[pc].size();
        if (!n) continue;
        DevTmp t_np, t_off, t_prim, t_Q;                         // freed on every return path
        RT_CUDA(cudaMalloc(&t_np.p, n * sizeof(int)));
        RT_CUDA(cudaMalloc(&t_off.p, n * sizeof(int)));
        RT_CUDA(cudaMalloc(&t_prim.p, rows[pc].size() * sizeof(double)));
        RT_CUDA(cudaMalloc(&t_Q.p, n * sizeof(double)));
        int *d_np = (int*)t_np.p, *d_off = (int*)t_off.p;
        double *d_prim = (double*)t_prim.p, *d_Q = (double*)t_Q.p;
        RT_CUDA(cudaMemcpyAsync(d_np, cand_np[pc].data(), n * sizeof(int), cudaMemcpyHostToDevice, st));
        RT_CUDA(cudaMemcpyAsync(d_off, cand_off[pc].data(), n * sizeof(int), cudaMemcpyHostToDevice, st));
        RT_CUDA(cudaMemcpyAsync(d_prim, rows[pc].data(), rows[pc].size() * sizeof(double), cudaMemcpyHostToDevice, st));
        // pairs with a d shell take the general path (eri_generic.cu)
        const int pl1 = pairclass_l1(pc), pl2 = pairclass_l2(pc);
        if (pl1 > 1) RT_TRY(schwarz_general(pl1, pl2, n, d_np, d_off, d_prim, h->tabs.boys[2 * (pl1 + pl2)], d_Q, st));
        else RT_TRY(schwarz_device(pc, n, d_np, d_off, d_prim, h->tabs.boys[2 * pc], d_Q, st));
        h->kernel_launches++;
        std::vector<double> Q(n);
        RT_CUDA(cudaMemcpyAsync(Q.data(), d_Q, n * sizeof(double), cudaMemcpyDeviceToHost, st));
        RT_CUDA(cudaStreamSynchronize(st));
        for (int k = 0; k < n; ++k) pairs[cand_id[pc][k]].Q = Q[k];
        // primitive-level bounds: every primitive pair as a shell pair of its own, q_k = sqrt(max (kk|kk))
        const int nrow = (int)(rows[pc].size() / PRIM_STRIDE);
        std::vector<int> one(nrow, 1), idx(nrow);
        std::iota(idx.begin(), idx.end(), 0);
        DevTmp t_np1, t_off1, t_Q1;
        RT_CUDA(cudaMalloc(&t_np1.p, nrow * sizeof(int)));
        RT_CUDA(cudaMalloc(&t_off1.p, nrow * sizeof(int)));
        RT_CUDA(cudaMalloc(&t_Q1.p, nrow * sizeof(double)));
        RT_CUDA(cudaMemcpyAsync(t_np1.p, one.data(), nrow * sizeof(int), cudaMemcpyHostToDevice, st));
        RT_CUDA(cudaMemcpyAsync(t_off1.p, idx.data(), nrow * sizeof(int), cudaMemcpyHostToDevice, st));
        if (pl1 > 1) RT_TRY(schwarz_general(pl1, pl2, nrow, (int*)t_np1.p, (int*)t_off1.p, d_prim, h->tabs.boys[2 * (pl1 + pl2)], (double*)t_Q1.p, st));
        else RT_TRY(schwarz_device(pc, nrow, (int*)t_np1.p, (int*)t_off1.p, d_prim, h->tabs.boys[2 * pc], (double*)t_Q1.p, st));
        h->kernel_launches++;
        qprim[pc].resize(nrow);
        RT_CUDA(cudaMemcpyAsync(qprim[pc].data(), t_Q1.p, nrow * sizeof(double), cudaMemcpyDeviceToHost, st));
        RT_CUDA(cudaStreamSynchronize(st));
    }
    double Qmax = 0.0;
    for (const Pair& P : pairs) Qmax = std::max(Qmax, P.Q);
    RT_CHECK(Qmax > 0.0 && std::isfinite(Qmax), "Schwarz bounds are not finite/positive");
    const double tau = h->tau;

    // ---- primitive screening: a primitive pair k whose own bound q_k cannot lift any integral above tau_p
    // (q_k Q_max < tau_p, tau_p = min(1e-3 tau, 1e-15); |(k.|cd)| <= q_k Q_cd) is dropped from its shell pair, and the pair moves to the contraction
    // sub-class of what is left (9 -> 6 -> 3 -> 1 primitive pairs; kept rows in order of descending bound).  The Schwarz bound Q
    // of the shell pair, hence the R14 quartet set, is untouched; the neglected primitive quartets are a thousand
    // times smaller than what the shell-level screening drops.  tau = 0 keeps every primitive.
    const double tau_p = prim_threshold(tau);
    for (Pair& P : pairs) {
        std::vector<int> order(P.np);
        std::iota(order.begin(), order.end(), 0);
        std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return qprim[P.pc][P.row + x] > qprim[P.pc][P.row + y]; });
        int neff = 0;
        for (int k = 0; k < P.np; ++k) neff += (qprim[P.pc][P.row + k] * Qmax >= tau_p) ? 1 : 0;
        neff = std::max(neff, 1);
        const int nstore = neff <= 1 ? 1 : (neff <= 3 ? 3 : (neff <= 6 ? 6 : 9));
        if (nstore < P.np) {
            order.resize(nstore);
            P.np = nstore;
            P.sub = np_to_sub(nstore);
        }
        P.sel = order;                      // most significant primitive first: quartet-level prefixes (jk_eval.cu)
    }

    // ---- keep, classify, sort by bound
    std::vector<int> cls[NKETCLASS];
    for (int k = 0; k < (int)pairs.size(); ++k) {
        const Pair& P = pairs[k];
        if (!(P.Q > 0.0) || P.Q * Qmax < tau) continue;
        cls[P.pc * NSUB + P.sub].push_back(k);
    }
    long long nkept = 0;
    std::vector<std::vector<double>> hQ(NKETCLASS);
    for (int kc = 0; kc < NKETCLASS; ++kc) {
        std::vector<int>& v = cls[kc];
        std::sort(v.begin(), v.end(), [&](int x, int y) {
            if (pairs[x].Q != pairs[y].Q) return pairs[x].Q > pairs[y].Q;
            return x < y;
        });
        const int n = (int)v.size(), np = sub_to_np(kc % NSUB), pc = kc / NSUB;
        nkept += n;
        std::vector<double> soa((size_t)np * PRIM_STRIDE * std::max(n, 1), 0.0);
        std::vector<double> aos((size_t)np * PRIM_STRIDE * std::max(n, 1), 0.0);
        std::vector<int> aoc(std::max(n, 1), 0), aod(std::max(n, 1), 0), same(std::max(n, 1), 0);
        std::vector<float> qsoa((size_t)np * std::max(n, 1), 0.f), qaos((size_t)np * std::max(n, 1), 0.f);
        hQ[kc].assign(std::max(n, 1), 0.0);
        for (int q = 0; q < n; ++q) {
            Pair& P = pairs[v[q]];
            P.pos = q;
            hQ[kc][q] = P.Q;
            aoc[q] = H.ao[P.s1]; aod[q] = H.ao[P.s2]; same[q] = (P.s1 == P.s2);
            for (int k = 0; k < np; ++k) {
                // float is enough for a screening bound; rounded up so that it never under-estimates
                const float qf = std::nextafter((float)(qprim[pc][P.row + P.sel[k]] * (1.0 + 1e-6)), INFINITY);
                qsoa[(size_t)k * n + q] = qf;
                qaos[(size_t)q * np + k] = qf;
            }
            for (int k = 0; k < np; ++k)
                for (int f = 0; f < PRIM_STRIDE; ++f)
                {
                    soa[((size_t)k * PRIM_STRIDE + f) * n + q] = rows[pc][(size_t)(P.row + P.sel[k]) * PRIM_STRIDE + f];
                    aos[((size_t)q * np + k) * PRIM_STRIDE + f] = rows[pc][(size_t)(P.row + P.sel[k]) * PRIM_STRIDE + f];
                }
        }
        KetClass& K = h->tabs.kets[kc];
        K.n = n; K.np = np;
        RT_TRY(upload(h, hQ[kc], &K.Q));
        RT_TRY(upload(h, aoc, &K.ao_c));
        RT_TRY(upload(h, aod, &K.ao_d));
        RT_TRY(upload(h, same, &K.same));
        RT_TRY(upload(h, soa, &K.prim));
        RT_TRY(upload(h, aos, &K.prim_aos));
        RT_TRY(upload(h, qsoa, &K.qp));
        RT_TRY(upload(h, qaos, &K.qp_aos));
    }

    // ---- ordered bra records grouped into a-lists keyed by (shell a, l_b, sub)
    struct Rec { int a, b, pair, canonical; };
    std::map<std::tuple<int, int, int>, std::vector<Rec>> groups;
    for (int kc = 0; kc < NKETCLASS; ++kc)
        for (int k : cls[kc]) {
            const Pair& P = pairs[k];
            groups[{P.s1, H.l[P.s2], P.sub}].push_back({P.s1, P.s2, k, 1});
            if (P.s1 != P.s2) groups[{P.s2, H.l[P.s1], P.sub}].push_back({P.s2, P.s1, k, 0});
        }
    std::vector<BraRec> recs, jrecs;
    std::vector<AList> alists;
    std::vector<int> alist_la, alist_lb;
    for (auto& g : groups) {
        std::vector<Rec>& v = g.second;
        std::sort(v.begin(), v.end(), [&](const Rec& x, const Rec& y) { return pairs[x.pair].pos < pairs[y.pair].pos; });
        AList al;
        al.ao_a = H.ao[std::get<0>(g.first)];
        al.rec_begin = (int)recs.size();
        al.jrec_begin = (int)jrecs.size();
        al.ketclass = pairs[v[0].pair].pc * NSUB + pairs[v[0].pair].sub;
        al.np = pairs[v[0].pair].np;
        al.Qmax = pairs[v[0].pair].Q;
        for (const Rec& r : v) {
            const Pair& P = pairs[r.pair];
            BraRec br;
            br.Q = P.Q; br.ao_b = H.ao[r.b]; br.pos = P.pos;
            br.flags = (r.canonical ? 1 : 0) | (r.a == r.b ? 2 : 0);
            br.pad = 0;
            recs.push_back(br);
            if (r.canonical) jrecs.push_back(br);
        }
        al.rec_end = (int)recs.size();
        al.jrec_end = (int)jrecs.size();
        alists.push_back(al);
        alist_la.push_back(H.l[std::get<0>(g.first)]);
        alist_lb.push_back(std::get<1>(g.first));
    }
    RT_TRY(upload(h, recs, &h->tabs.recs));
    RT_TRY(upload(h, jrecs, &h->tabs.jrecs));
    RT_TRY(upload(h, alists, &h->tabs.alists));
    h->tabs.tau = tau;
    h->tabs.nao = h->nao;

    // ---- segments (bra pair class x ket pair class, unique quartets), their staging-buffer maps and the
    //      evaluation / digestion work lists
    // pairs q of class kc (Q sorted descending) with Q_q * Qother >= tau: the SAME product test the kernels apply
    // per lane, so that the staging map and the kernels agree on which batches exist down to the last bit
    auto count_prod_ge = [&](int kc, double Qother) {
        const std::vector<double>& q = hQ[kc];
        const int n = h->tabs.kets[kc].n;
        int lo = 0, hi = n;                         // first index whose product falls below tau
        while (lo < hi) {
            const int mid = (lo + hi) / 2;
            if (q[mid] * Qother >= tau) lo = mid + 1; else hi = mid;
        }
        return lo;
    };
    auto nkets_of = [&](int kc_ket, double Qp) {    // kets q (a prefix of the list) with Qp Q_q >= tau
        return tau > 0.0 ? count_prod_ge(kc_ket, Qp) : h->tabs.kets[kc_ket].n;
    };
    double n_eval = 0, nprim_eval = 0, fl_eval = 0;
    size_t buf_need = 1;
    h->launches.clear();
    h->segments.clear();
    for (int kcb = NKETCLASS - 1; kcb >= 0; --kcb)
        for (int kck = NKETCLASS - 1; kck >= 0; --kck) {
            const int pcb = kcb / NSUB, pck = kck / NSUB;
            // unique quartets: higher pair type is the bra; within a type the lower class id; within a class p <= q
            if (pck > pcb || (pck == pcb && kcb > kck)) continue;
            const int nb = h->tabs.kets[kcb].n, nk = h->tabs.kets[kck].n;
            if (nb == 0 || nk == 0) continue;
            const bool same = (kcb == kck);
            Segment sg{};
            sg.kc_bra = kcb; sg.kc_ket = kck;
            sg.la = pairclass_l1(pcb); sg.lb = pairclass_l2(pcb); sg.lc = pairclass_l1(pck); sg.ld = pairclass_l2(pck);
            sg.ni = ncart(sg.la) * ncart(sg.lb) * ncart(sg.lc) * ncart(sg.ld);
            // staging map: pair p owns the 32-ket batches covering kets [same ? p : 0, nk_p)
            std::vector<long long> base(nb, 0);
            long long nbatch = 0, nquart = 0;
            for (int p = 0; p < nb; ++p) {
                base[p] = nbatch;
                const int nkp = nkets_of(kck, hQ[kcb][p]);
                const int lo = same ? p : 0;
                if (nkp > lo) {
                    nbatch += ((nkp - 1) >> 5) - (lo >> 5) + 1;
                    nquart += nkp - lo;
                }
            }
            sg.nbatch = nbatch; sg.nquartets = nquart;
            if (nquart == 0) continue;
            n_eval += (double)nquart;
            nprim_eval += (double)nquart * h->tabs.kets[kcb].np * h->tabs.kets[kck].np;
            fl_eval += (double)nquart * h->tabs.kets[kcb].np * h->tabs.kets[kck].np * flops_prim(sg.la, sg.lb, sg.lc, sg.ld);
            buf_need = std::max(buf_need, (size_t)nbatch * sg.ni * 32);
            sg.incore_off = h->eri_all_need;
            h->eri_all_need += (size_t)nbatch * sg.ni * 32;
            RT_TRY(upload(h, base, &sg.batch_base));
            // evaluation blocks: JK_BLOCK kets x a run of bra pairs (rows staged in shared memory)
            const int npb = h->tabs.kets[kcb].np;
            // at most 32 bra pairs per block: shallow contractions (1 or 3 primitive pairs) would otherwise give a
            // handful of very long blocks per segment and leave SMs idle
            // general path (classes with a d shell, eri_generic.cu): a block is 32 kets x 4 component workers and walks
            // few bra pairs, so that even a handful of d shells spreads over many blocks (at most ~2e5 blocks per segment)
            const bool general = segment_is_general(sg);
            const int kstep = general ? 32 : JK_BLOCK;
            const int G = general ? (int)std::max<long long>(1, ((long long)nb * ((nk + 31) / 32) + 199999) / 200000)
                                  : std::min(32, std::min(JK_BLOCK, EVAL_MAX_ROWS / npb));
            std::vector<EvalItem> items;
            for (int k0 = 0; k0 < nk; k0 += kstep) {
                int hi = tau > 0.0 ? count_prod_ge(kcb, hQ[kck][k0]) : nb;     // bra pairs reaching this chunk
                if (same) hi = std::min(hi, std::min(nb, k0 + kstep));
                for (int p0 = 0; p0 < hi; p0 += G) items.push_back(EvalItem{k0, p0, std::min(hi, p0 + G)});
            }
            sg.nitems = (int)items.size();
            RT_TRY(upload(h, items, &sg.items));
            // digestion launches: ordered bra classes (a-lists) of this bra pair class against the ket class
            sg.first_launch = (int)h->launches.size();
            for (int orient = 0; orient < 2; ++orient) {
                if (!digest_has_alist_kernels(sg)) break;          // large d classes: one general kernel digests the whole segment
                if (orient == 1 && sg.la == sg.lb) break;          // ss and pp pairs: one ordered class
                const int la = orient == 0 ? sg.la : sg.lb, lb = orient == 0 ? sg.lb : sg.la;
                std::vector<std::pair<double, WorkItem>> witems;
                for (int ai = 0; ai < (int)alists.size(); ++ai) {
                    if (alist_la[ai] != la || alist_lb[ai] != lb || alists[ai].ketclass != kcb) continue;
                    const AList& al = alists[ai];
                    const int nkmax = nkets_of(kck, al.Qmax);
                    const int q0 = same ? (recs[al.rec_begin].pos / JK_BLOCK) * JK_BLOCK : 0;
                    const double len = al.rec_end - al.rec_begin;
                    for (int k0 = q0; k0 < nkmax; k0 += JK_BLOCK) witems.push_back({len, WorkItem{ai, k0}});
                }
                std::stable_sort(witems.begin(), witems.end(), [](const auto& x, const auto& y) { return x.first > y.first; });
                std::vector<WorkItem> w;
                w.reserve(witems.size());
                for (auto& it : witems) w.push_back(it.second);
                JKLaunch L{};
                L.la = la; L.lb = lb; L.lc = sg.lc; L.ld = sg.ld; L.ketclass = kck;
                L.seg = (int)h->segments.size();
                L.nwork = (int)w.size();
                RT_TRY(upload(h, w, &L.work));
                h->launches.push_back(L);
            }
            sg.nlaunch = (int)h->launches.size() - sg.first_launch;
            h->segments.push_back(sg);
        }
    h->eri_buf_need = buf_need;

    // ---- R14 counts: unique quartets with Q_ab Q_cd >= tau, and the flop model on them
    {
        double ordered = 0, ordered_prim = 0, diag = 0, diag_prim = 0, fl_ord = 0, fl_diag = 0, nint_ord = 0, nint_diag = 0;
        // primitive counts as GIVEN (a padded 2-primitive shell counts 2): prefix sums over each sorted class list
        std::vector<std::vector<double>> pre(NKETCLASS);
        for (int kc = 0; kc < NKETCLASS; ++kc) {
            pre[kc].assign(cls[kc].size() + 1, 0.0);
            for (size_t q = 0; q < cls[kc].size(); ++q) pre[kc][q + 1] = pre[kc][q] + pairs[cls[kc][q]].np_true;
        }
        for (int kc1 = 0; kc1 < NKETCLASS; ++kc1)
            for (int k : cls[kc1]) {
                const Pair& P = pairs[k];
                const int l1 = pairclass_l1(P.pc), l2 = pairclass_l2(P.pc);
                for (int kc2 = 0; kc2 < NKETCLASS; ++kc2) {
                    const int n2 = tau > 0.0 ? count_prod_ge(kc2, P.Q) : h->tabs.kets[kc2].n;
                    const int pc2 = kc2 / NSUB, l3 = pairclass_l1(pc2), l4 = pairclass_l2(pc2);
                    const double npq = (double)P.np_true * pre[kc2][n2];       // primitive quartets of these n2 quartets
                    ordered += n2;
                    ordered_prim += npq;
                    fl_ord += npq * flops_prim(l1, l2, l3, l4);
                    nint_ord += (double)n2 * ncart(l1) * ncart(l2) * ncart(l3) * ncart(l4);
                }
                if (P.Q * P.Q >= tau) {
                    diag += 1; diag_prim += (double)P.np_true * P.np_true;
                    fl_diag += (double)P.np_true * P.np_true * flops_prim(l1, l2, l1, l2);
                    nint_diag += (double)ncart(l1) * ncart(l2) * ncart(l1) * ncart(l2);
                }
            }
        h->info[RTTDA_INFO_NQUARTETS] = 0.5 * (ordered + diag);
        h->info[RTTDA_INFO_NPRIM_QUARTETS] = 0.5 * (ordered_prim + diag_prim);
        (void)fl_ord; (void)fl_diag;
        h->info[RTTDA_INFO_FLOPS_EVAL] = fl_eval;   // on the primitive quartets the kernels evaluate (after primitive screening)
        h->info[RTTDA_INFO_FLOPS_DIGEST_PER_VEC] = 20.0 * 0.5 * (nint_ord + nint_diag);
    }
    h->info[RTTDA_INFO_NPAIRS_TOTAL] = (double)npairs_total;
    h->info[RTTDA_INFO_NPAIRS_KEPT] = (double)nkept;
    h->info[RTTDA_INFO_NQUARTETS_EVAL] = n_eval;
    h->info[RTTDA_INFO_NPRIM_EVAL] = nprim_eval;
    h->info[RTTDA_INFO_JK_LAUNCHES] = (double)h->launches.size();
    h->info[RTTDA_INFO_QMAX] = Qmax;
    h->info[RTTDA_INFO_NVEC_CHUNK] = 0.0;
    h->info[RTTDA_INFO_ERI_BUF_BYTES] = (double)buf_need * sizeof(double);
    h->info[RTTDA_INFO_ERI_ALL_BYTES] = (double)h->eri_all_need * sizeof(double);

    // ---- MO coefficients, eps differences, dipoles
    auto dalloc = [&](double** p, size_t n) -> int {
        RT_CUDA(cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(double)));
        h->dev_allocs.push_back(*p);
        return RTTDA_OK;
    };
    const size_t no = h->nocc, nv = h->nvirt;
    RT_TRY(dalloc(&h->C_occ, N * no));
    RT_TRY(dalloc(&h->C_virt, N * nv));
    RT_CUDA(cudaMemcpyAsync(h->C_occ, C_occ, N * no * sizeof(double), cudaMemcpyDeviceToDevice, st));
    RT_CUDA(cudaMemcpyAsync(h->C_virt, C_virt, N * nv * sizeof(double), cudaMemcpyDeviceToDevice, st));
    std::vector<double> de(no * nv);
    for (size_t i = 0; i < no; ++i)
        for (size_t a = 0; a < nv; ++a) de[i * nv + a] = eps[no + a] - eps[i];
    RT_TRY(dalloc(&h->deps, no * nv));
    RT_CUDA(cudaMemcpyAsync(h->deps, de.data(), de.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    std::vector<double> D(3 * N * N);
    one_electron_host(H, nullptr, D.data());
    RT_TRY(dalloc(&h->D_ao, 3 * N * N));
    RT_CUDA(cudaMemcpyAsync(h->D_ao, D.data(), D.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    RT_TRY(dalloc(&h->D_oo, 3 * no * no));
    RT_TRY(dalloc(&h->D_vv, 3 * nv * nv));
    RT_TRY(dalloc(&h->D_ov, 3 * no * nv));
    DevTmp t_tmp;                               // D C_v | D C_o, [3][N][max(no,nv)]
    const size_t nm = std::max(no, nv);
    RT_CUDA(cudaMalloc(&t_tmp.p, 3 * N * nm * sizeof(double)));
    double* tmp = (double*)t_tmp.p;
    // tmp = D^k C_v ; D_vv = C_v^T tmp ; D_ov = C_o^T tmp ; then tmp = D^k C_o ; D_oo = C_o^T tmp
    GemmDesc g{};
    g.alpha = 1.0; g.beta = 0.0; g.batch = 3;
    g.M = (int)N; g.N = (int)nv; g.K = (int)N;
    g.A = h->D_ao; g.sam = N; g.sak = 1; g.sabatch = N * N;
    g.B = h->C_virt; g.sbk = nv; g.sbn = 1; g.sbbatch = 0;
    g.C = tmp; g.scm = nv; g.scn = 1; g.scbatch = N * nv;
    RT_TRY(gemm_f64(g, st));
    g.M = (int)nv; g.N = (int)nv; g.K = (int)N;
    g.A = h->C_virt; g.sam = 1; g.sak = nv; g.sabatch = 0;
    g.B = tmp; g.sbk = nv; g.sbn = 1; g.sbbatch = N * nv;
    g.C = h->D_vv; g.scm = nv; g.scn = 1; g.scbatch = nv * nv;
    RT_TRY(gemm_f64(g, st));
    g.M = (int)no; g.A = h->C_occ; g.sam = 1; g.sak = no;
    g.C = h->D_ov; g.scm = nv; g.scbatch = no * nv;
    RT_TRY(gemm_f64(g, st));
    g.M = (int)N; g.N = (int)no; g.K = (int)N;
    g.A = h->D_ao; g.sam = N; g.sak = 1; g.sabatch = N * N;
    g.B = h->C_occ; g.sbk = no; g.sbn = 1; g.sbbatch = 0;
    g.C = tmp; g.scm = no; g.scn = 1; g.scbatch = N * no;
    RT_TRY(gemm_f64(g, st));
    g.M = (int)no; g.N = (int)no; g.K = (int)N;
    g.A = h->C_occ; g.sam = 1; g.sak = no; g.sabatch = 0;
    g.B = tmp; g.sbk = no; g.sbn = 1; g.sbbatch = N * no;
    g.C = h->D_oo; g.scm = no; g.scn = 1; g.scbatch = no * no;
    RT_TRY(gemm_f64(g, st));
    h->kernel_launches += 5;
    std::vector<double> doo(3 * no * no);
    RT_CUDA(cudaMemcpyAsync(doo.data(), h->D_oo, doo.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
    RT_CUDA(cudaStreamSynchronize(st));
    // Dipole origin = electronic centroid of the ground state, c_k = tr(D_oo^k)/n_occ (R6): with orthonormal MOs the
    // shift r -> r - c is D_oo -> D_oo - c 1, D_vv -> D_vv - c 1, D_ov unchanged, and D_00 = 2 tr D_oo (R3: sum
    // over spin orbitals) becomes zero.  Without it D_00 grows with the molecule's distance from the coordinate
    // origin (1e4 au at 1280 AOs) and E(t) D_00 is a global phase no fixed-step propagator can follow.
    for (int k = 0; k < 3; ++k) {
        double tr = 0.0;
        for (size_t i = 0; i < no; ++i) tr += doo[k * no * no + i * no + i];
        const double c = tr / (double)no;
        shift_diag_kernel<<<(unsigned)((no + 255) / 256), 256, 0, st>>>((int)no, -c, h->D_oo + (size_t)k * no * no);
        shift_diag_kernel<<<(unsigned)((nv + 255) / 256), 256, 0, st>>>((int)nv, -c, h->D_vv + (size_t)k * nv * nv);
        double tr2 = 0.0;
        for (size_t i = 0; i < no; ++i) tr2 += doo[k * no * no + i * no + i] - c;
        h->D_00[k] = 2.0 * tr2;
    }
    RT_CUDA(cudaGetLastError());
    RT_CUDA(cudaStreamSynchronize(st));
    h->kernel_launches += 6;
    for (auto& e : h->ev) RT_CUDA(cudaEventCreate(&e));
    RT_CUDA(cudaMalloc((void**)&h->d_primcount, 8 * sizeof(unsigned long long)));
    h->dev_allocs.push_back(h->d_primcount);
    RT_CUDA(cudaMemsetAsync(h->d_primcount, 0, 8 * sizeof(unsigned long long), st));
    RT_CUDA(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
    for (int l = 0; l < Handle::MAXLANES; ++l) {
        RT_CUDA(cudaStreamCreateWithFlags(&h->lane_st[l], cudaStreamNonBlocking));
        RT_CUDA(cudaEventCreateWithFlags(&h->lane_ev[l], cudaEventDisableTiming));
    }
    {
        // all integrals of one pass below 8 GB: the kernels are small, run 8 lanes side by side; else the pipeline
        const char* e = getenv("RTTDA_LANES");
        const int nl = e ? atoi(e) : ((double)h->eri_all_need * sizeof(double) < 8e9 ? Handle::MAXLANES : 0);
        RT_TRY(assign_lanes(h, nl));
        h->use_graph = h->nlanes > 0;              // small molecules: launch-bound steps are replayed as a CUDA graph
    }
    h->info[RTTDA_INFO_CREATE_MS] =
        std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return RTTDA_OK;
}

// Deal the segments to `nlanes` lanes: longest estimated run time first, each onto the lane with the least work so far
// (cost model: flop model of the evaluation + 40 flop-equivalents per stored integral for the gather-bound digestion).
int assign_lanes(Handle* h, int nlanes)
{
    RT_CHECK(nlanes >= 0 && nlanes <= Handle::MAXLANES, "lanes must be in 0..8 (0 = two-buffer pipeline)");
    std::vector<std::pair<double, int>> cost;
    for (int i = 0; i < (int)h->segments.size(); ++i) {
        const Segment& sg = h->segments[i];
        if (sg.nitems == 0) continue;
        const double npq = (double)sg.nquartets * h->tabs.kets[sg.kc_bra].np * h->tabs.kets[sg.kc_ket].np;
        cost.push_back({npq * flops_prim(sg.la, sg.lb, sg.lc, sg.ld) + 40.0 * 6.0 * (double)sg.nquartets * sg.ni, i});
    }
    std::sort(cost.begin(), cost.end(), [](const auto& a, const auto& b) { return a.first > b.first; });
    double load[Handle::MAXLANES] = {0};
    for (int l = 0; l < Handle::MAXLANES; ++l) { h->lane_segs[l].clear(); h->lane_need[l] = 1; }
    for (const auto& c : cost) {
        int best = 0;
        for (int l = 1; l < nlanes; ++l) if (load[l] < load[best]) best = l;
        load[best] += c.first;
        h->lane_segs[best].push_back(c.second);
        const Segment& sg = h->segments[c.second];
        h->lane_need[best] = std::max(h->lane_need[best], (size_t)sg.nbatch * sg.ni * 32);
    }
    h->nlanes = nlanes;
    return RTTDA_OK;
}

int overlap_host(const rttda_basis_t* basis, int nao, double* S, double* D)
{
    HostBasis H;
    RT_TRY(load_basis(basis, H));
    RT_CHECK(H.nao == nao, "nao does not match the shell table");
    one_electron_host(H, S, D);
    return RTTDA_OK;
}

}  // namespace rttda
