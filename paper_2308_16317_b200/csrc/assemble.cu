// assemble.cu -- K1: device-side assembly of the KKR matrices M = t^{-1} - g0,
// "Further code acceleration is expected if the KKR matrix is constructed on GPUs".
//
//   g0_{LL'}(R) = -4 pi i kappa sum_{l''} i^{l-l'+l''} h_{l''}(kappa R) Y_{l'',m'-m}(R^) C(L,L',L'')
//   (DESIGN.md "Readings" A1-A4).
//
// Gaunt numbers come from the closed form (two Wigner 3j symbols, Racah's sum) -- a different
// route from the oracle's quadrature.  HBM-write-bound: 16 n^2 bytes per item.
#include "common.cuh"
#include "internal.h"

namespace lsms {

// ---------------------------------------------------------------- Gaunt numbers, closed form

__host__ __device__ inline double fact(int n) { double f = 1.0; for (int i = 2; i <= n; ++i) f *= (double)i; return f; }

// Wigner 3j symbol (j1 j2 j3; m1 m2 m3), integer arguments, Racah's formula.
__host__ __device__ double wigner3j(int j1, int j2, int j3, int m1, int m2, int m3) {
    if (m1 + m2 + m3 != 0) return 0.0;
    if (j3 < abs(j1 - j2) || j3 > j1 + j2) return 0.0;
    if (abs(m1) > j1 || abs(m2) > j2 || abs(m3) > j3) return 0.0;
    double delta = fact(j1 + j2 - j3) * fact(j1 - j2 + j3) * fact(-j1 + j2 + j3) / fact(j1 + j2 + j3 + 1);
    double pre = sqrt(delta * fact(j1 + m1) * fact(j1 - m1) * fact(j2 + m2) * fact(j2 - m2) * fact(j3 + m3) * fact(j3 - m3));
    int tmin = 0;
    if (j2 - j3 - m1 > tmin) tmin = j2 - j3 - m1;
    if (j1 - j3 + m2 > tmin) tmin = j1 - j3 + m2;
    int tmax = j1 + j2 - j3;
    if (j1 - m1 < tmax) tmax = j1 - m1;
    if (j2 + m2 < tmax) tmax = j2 + m2;
    double s = 0.0;
    for (int t = tmin; t <= tmax; ++t) {
        double d = fact(t) * fact(j3 - j2 + t + m1) * fact(j3 - j1 + t - m2) * fact(j1 + j2 - j3 - t) * fact(j1 - t - m1) * fact(j2 - t + m2);
        s += ((t & 1) ? -1.0 : 1.0) / d;
    }
    int ph = j1 - j2 - m3;
    return ((ph & 1) ? -1.0 : 1.0) * pre * s;
}

// C(L,L',L'') = Int Y_L^* Y_L' Y_L''^* dOmega, m'' = m' - m.
__host__ __device__ double gaunt_closed_form(int l, int m, int lp, int mp, int lpp) {
    int mpp = mp - m;
    if (abs(mpp) > lpp || ((l + lp + lpp) & 1)) return 0.0;
    const double FOUR_PI = 12.566370614359172953850573533118;
    double pref = sqrt((2.0 * l + 1.0) * (2.0 * lp + 1.0) * (2.0 * lpp + 1.0) / FOUR_PI);
    double v = pref * wigner3j(l, lp, lpp, 0, 0, 0) * wigner3j(l, lp, lpp, -m, mp, -mpp);
    return ((m + mpp) & 1) ? -v : v;
}

double gaunt_closed_form_host(int l, int m, int lp, int mp, int lpp) { return gaunt_closed_form(l, m, lp, mp, lpp); }

__host__ __device__ inline void l_m_of(int L, int& l, int& m) { l = 0; while ((l + 1) * (l + 1) <= L) ++l; m = L - l * (l + 1); }

// Table entry t (0..lmax) of the pair (L,L'), stored at [(t*kmax + L')*kmax + L]:
//   coef = -4 pi i * i^{l-l'+l''} * C(L,L',L''),  idx = L'' = l''(l''+1) + m' - m,  l'' = |l-l'| + 2t.
__device__ __forceinline__ void legendre_table_block(int l2, double* __restrict__ leg);

// The LAST block of the grid fills the Legendre recurrence table (below) instead: one launch for both tables.
__global__ void k_gaunt_table(int lmax, c128* __restrict__ coef, int* __restrict__ idx, double* __restrict__ leg) {
    if (blockIdx.x == gridDim.x - 1) { legendre_table_block(2 * lmax, leg); return; }
    int kmax = (lmax + 1) * (lmax + 1), nt = lmax + 1;
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= kmax * kmax * nt) return;
    int L = e % kmax, Lp = (e / kmax) % kmax, t = e / (kmax * kmax);
    int l, m, lp, mp; l_m_of(L, l, m); l_m_of(Lp, lp, mp);
    int lpp = abs(l - lp) + 2 * t, mpp = mp - m;
    c128 c = cmake(0.0, 0.0); int id = 0;
    if (lpp <= l + lp && abs(mpp) <= lpp) {
        double g = gaunt_closed_form(l, m, lp, mp, lpp);
        const double FOUR_PI = 12.566370614359172953850573533118;
        // -4 pi i * i^p,  p = l - l' + l'' >= 0:  i^(p+1) * (-4 pi)
        int p = (l - lp + lpp + 1) & 3;
        double v = -FOUR_PI * g;
        c = (p == 0) ? cmake(v, 0.0) : (p == 1) ? cmake(0.0, v) : (p == 2) ? cmake(-v, 0.0) : cmake(0.0, -v);
        id = lpp * (lpp + 1) + mpp;
    }
    coef[e] = c; idx[e] = id;
}

// ---------------------------------------------------------------- t^{-1} from phase shifts

__device__ inline c128 csqrt_upper(c128 z) {       // principal root with Im >= 0 for Im z >= 0
    double r = hypot(z.x, z.y);
    c128 k;
    if (r == 0.0) return cmake(0.0, 0.0);
    if (z.x >= 0.0) { double t = sqrt(0.5 * (r + z.x)); k = cmake(t, z.y / (2.0 * t)); }
    else { double t = sqrt(0.5 * (r - z.x)); k = cmake(fabs(z.y) / (2.0 * t), copysign(t, z.y)); }
    if (k.y < 0.0) k = cneg(k);
    return k;
}

// Reading A4 / include/lsms_tau.h: illegal input VALUES are reported per item (first non-zero code wins, no sync):
//   -4 z non-finite or Im z < 0,  -2 species index out of range,  -1 phase shift non-finite or sin(delta) = 0.
__device__ __forceinline__ bool finite2(c128 a) { return isfinite(a.x) && isfinite(a.y); }

__global__ void k_tinv(const c128* __restrict__ delta, const int* __restrict__ species, const c128* __restrict__ z,
                       int lmax, int n_sites, int nspin, int n_species, int batch, c128* __restrict__ tinv, c128* __restrict__ kappa,
                       int* __restrict__ info) {
    int nl = lmax + 1;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long total = (long long)batch * n_sites * nspin * nl;
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    if (e < batch) {
        const c128 zz = z[e];
        const bool bad = !finite2(zz) || zz.y < 0.0;
        kappa[e] = bad ? cmake(qnan, qnan) : csqrt_upper(zz);
        if (bad) atomicCAS(&info[e], 0, -4);
    }
    if (e >= total) return;
    int l = (int)(e % nl); long long r = e / nl;
    int s = (int)(r % nspin); r /= nspin;
    int site = (int)(r % n_sites); int b = (int)(r / n_sites);
    const c128 zz = z[b];
    const bool zbad = !finite2(zz) || zz.y < 0.0;
    const int sp = species[(size_t)b * n_sites + site];
    if (sp < 0 || sp >= n_species) { atomicCAS(&info[b], 0, -2); tinv[e] = cmake(qnan, qnan); return; }
    c128 kap = csqrt_upper(zz);
    c128 d = delta[((size_t)sp * nspin + s) * nl + l];
    // sin(a+ib) = sin a cosh b + i cos a sinh b ;  e^{i(a+ib)} = e^{-b}(cos a + i sin a)
    double sa, ca; sincos(d.x, &sa, &ca);
    double eb = exp(-d.y);
    c128 sn = cmake(sa * cosh(d.y), ca * sinh(d.y));
    c128 ex = cmake(eb * ca, eb * sa);
    c128 t = cneg(cdiv(kap, cmul(sn, ex)));       // -kappa / (sin d e^{i d})
    if (!zbad && (!finite2(d) || !finite2(t))) atomicCAS(&info[b], 0, -1);
    tinv[e] = zbad ? cmake(qnan, qnan) : t;
}

// ---------------------------------------------------------------- Legendre recurrence table
// Fully normalised recurrence  Pbar_lm = a_lm (x Pbar_{l-1,m} - b_lm Pbar_{l-2,m}),
// Pbar_mm = d_m sin(theta) Pbar_{m-1,m-1}; a, b, d tabulated once so that K1 has no sqrt/div inside.
//   leg[0*S + l*(l2+1)+m] = a_lm, leg[1*S + ...] = b_lm, leg[2*S + m] = d_m,  S = (l2+1)^2
__device__ __forceinline__ void legendre_table_block(int l2, double* __restrict__ leg) {
    const int S = (l2 + 1) * (l2 + 1);
    for (int e = threadIdx.x; e < S; e += blockDim.x) {
        const int l = e / (l2 + 1), m = e % (l2 + 1);
        double a = 0.0, b = 0.0;
        if (l > m) {
            a = sqrt((4.0 * l * l - 1.0) / ((double)l * l - (double)m * m));
            b = sqrt((((double)l - 1.0) * (l - 1.0) - (double)m * m) / (4.0 * (l - 1.0) * (l - 1.0) - 1.0));
        }
        leg[e] = a; leg[S + e] = b;
        if (l == 0) leg[2 * S + m] = (m > 0) ? -sqrt((2.0 * m + 1.0) / (2.0 * m)) : 1.0;
    }
}

// ---------------------------------------------------------------- K1: column-strip assembly
// One CTA per (column site sj, item b): it writes the k full columns of M that belong to site sj,
// i.e. n*16 B contiguous per column (HBM-write-bound).
//   phase 1 (a1): one thread per row site si != sj builds hY[si][L''] = h_{l''}(kappa R) Y_{L''}(R^) in smem
//   phase 2 (a2): one thread per (L, L') pair of the site block walks the row sites of the chunk:
//                 -g0 = sum_t (-kappa coef_t) hY[idx_t]   (s == s'),  0 (s != s'),  t^{-1} on the site diagonal.
// Row sites are processed in chunks that fit shared memory.
constexpr int ASM_THREADS = 256;

template <int MAXNT, bool REP>   // MAXNT >= l_max + 1: length of the per-thread Gaunt term arrays; REP: shared-g0 mode (n_rep >= 1 items per CTA)
__global__ void __launch_bounds__(ASM_THREADS)
k_assemble(const c128* __restrict__ tinv, const double* __restrict__ site_pos, const double* __restrict__ moment,
           const c128* __restrict__ kappa, const c128* __restrict__ coef, const int* __restrict__ idx,
           const double* __restrict__ leg, int lmax, int n_sites, int canted, int chunk, int n_rep, int rep_stride,
           c128* __restrict__ Mout, int* __restrict__ info) {
    extern __shared__ __align__(16) unsigned char asm_smem[];
    const int kmax = (lmax + 1) * (lmax + 1), nt = lmax + 1, l2 = 2 * lmax, nl2 = (l2 + 1) * (l2 + 1);
    const int nspin = canted ? 2 : 1, k = kmax * nspin, kk2 = kmax * kmax, S = nl2;
    const size_t n = (size_t)n_sites * k;
    const int b = blockIdx.y, sj = blockIdx.x, tid = threadIdx.x;
    c128* hY = reinterpret_cast<c128*>(asm_smem);                 // [chunk][nl2]
    c128* M = Mout + (size_t)b * n * n;          // item b; items b + a*rep_stride, a < n_rep, share its geometry and kappa
    const size_t rep_elems = (size_t)rep_stride * n * n;
    const int nrep = REP ? n_rep : 1;
    const size_t c0 = (size_t)(sj == 0 ? n_sites - 1 : sj - 1) * k;
    // reading A4: Im kappa < 0 (the wrong sheet: h_l would grow with R) or a non-finite kappa rejects the item:
    // info = -5 and the whole matrix becomes NaN (kappa := NaN poisons every g0 and, below, every t^{-1} entry)
    c128 kap = kappa[b];
    const bool kbad = !(isfinite(kap.x) && isfinite(kap.y)) || kap.y < 0.0;
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    if (kbad) {
        kap = cmake(qnan, qnan);
        if (sj == 0) for (int a = tid; a < nrep; a += ASM_THREADS) atomicCAS(&info[(size_t)b + (size_t)a * rep_stride], 0, -5);
    }
    const c128 zero = kbad ? cmake(qnan, qnan) : cmake(0.0, 0.0);     // also the "zero" entries of a rejected item
    const double* pj = site_pos + ((size_t)b * n_sites + sj) * 3;
    const double xj = pj[0], yj = pj[1], zj = pj[2];

    for (int s0 = 0; s0 < n_sites; s0 += chunk) {
        const int ns = min(chunk, n_sites - s0);
        __syncthreads();
        // ---- phase 1: per-R tables
        for (int q = tid; q < ns; q += ASM_THREADS) {
            const int si = s0 + q;
            if (si == sj) continue;
            const double* pi = site_pos + ((size_t)b * n_sites + si) * 3;
            const double Rx = pi[0] - xj, Ry = pi[1] - yj, Rz = pi[2] - zj;
            const double R = sqrt(Rx * Rx + Ry * Ry + Rz * Rz);
            c128* out = hY + (size_t)q * nl2;
            // Y_lm(R^) by columns m (both signs), l = m..l2
            const double ct = Rz / R, rho = sqrt(Rx * Rx + Ry * Ry), st = rho / R;
            double cphi = 1.0, sphi = 0.0;
            if (rho > 0.0) { cphi = Rx / rho; sphi = Ry / rho; }
            double pmm = 0.28209479177387814347403972578039, er = 1.0, ei = 0.0;
            for (int m = 0; m <= l2; ++m) {
                if (m > 0) {
                    pmm *= leg[2 * S + m] * st;
                    const double t = er * cphi - ei * sphi; ei = er * sphi + ei * cphi; er = t;
                }
                double p2 = 0.0, p1 = pmm;
                for (int l = m; l <= l2; ++l) {
                    double pv = pmm;
                    if (l > m) { pv = leg[l * (l2 + 1) + m] * (ct * p1 - leg[S + l * (l2 + 1) + m] * p2); p2 = p1; p1 = pv; }
                    const c128 y = cmake(pv * er, pv * ei);
                    out[l * (l + 1) + m] = y;
                    if (m > 0) out[l * (l + 1) - m] = (m & 1) ? cmake(-y.x, y.y) : cmake(y.x, -y.y);   // (-1)^m conj
                }
            }
            // h_l(kappa R), l = 0..l2, multiplied in
            const c128 x = cscale(R, kap);
            double sn, cs; sincos(x.x, &sn, &cs);
            const double ed = exp(-x.y);
            const c128 eix = cmake(ed * cs, ed * sn);
            const c128 xinv = crecip(x);
            c128 h0 = cmul(cmake(0.0, -1.0), cmul(eix, xinv));                                        // -i e^{ix}/x
            c128 h1 = cneg(cmul(cadd(cmake(1.0, 0.0), cmul(cmake(0.0, 1.0), xinv)), cmul(eix, xinv)));   // -(1+i/x) e^{ix}/x
            for (int l = 0; l <= l2; ++l) {
                c128 h = (l == 0) ? h0 : h1;
                if (l >= 2) { h = csub(cscale((double)(2 * l - 1), cmul(xinv, h1)), h0); h0 = h1; h1 = h; }
                for (int e = l * l; e < (l + 1) * (l + 1); ++e) out[e] = cmul(h, out[e]);
            }
        }
        __syncthreads();
        // ---- phase 2: one thread per (L, L') pair of the site block; its Gaunt terms (pre-multiplied by -kappa) stay
        // in registers while it walks the row sites of the chunk: per element <= l_max+1 LDS.128 + complex FMAs and
        // one (canted: four) coalesced store -- consecutive threads hold consecutive L = consecutive rows.
        for (int p0 = 0; p0 < kk2; p0 += ASM_THREADS) {
            const int p = p0 + tid;
            if (p < kk2) {
                const int L = p % kmax, Lp = p / kmax;
                c128 cf[MAXNT]; int ix[MAXNT]; bool nz[MAXNT];
#pragma unroll
                for (int t = 0; t < MAXNT; ++t) {
                    nz[t] = false; cf[t] = zero; ix[t] = 0;
                    if (t < nt) {
                        const c128 c = coef[t * kk2 + Lp * kmax + L];
                        nz[t] = (c.x != 0.0 || c.y != 0.0);
                        cf[t] = cneg(cmul(kap, c));
                        ix[t] = idx[t * kk2 + Lp * kmax + L];
                    }
                }
                int lL = 0; while ((lL + 1) * (lL + 1) <= L) ++lL;
                c128* colp = M + n * (c0 + Lp) + L;                    // column (sj, spin 0, L'), row offset L
                for (int q = 0; q < ns; ++q) {
                    const int si = s0 + q;
                    const size_t rowb = (size_t)(si == 0 ? n_sites - 1 : si - 1) * k;
                    if (si != sj) {
                        const c128* hy = hY + (size_t)q * nl2;
                        c128 g = zero;
#pragma unroll
                        for (int t = 0; t < MAXNT; ++t) if (nz[t]) cfma(g, cf[t], hy[ix[t]]);
                        // g0 depends on the geometry and kappa only: one evaluation serves every item that shares them
                        for (int a = 0; a < nrep; ++a) {
                            c128* cp = colp + (size_t)a * rep_elems;
                            cp[rowb] = g;
                            if (canted) {
                                cp[rowb + kmax] = zero;                                   // (down, up)
                                cp[rowb + n * kmax] = zero;                               // (up, down)
                                cp[rowb + n * kmax + kmax] = g;                           // (down, down): g0 (x) 1_2
                            }
                        }
                    } else {
                        // site-diagonal block: t^{-1} (g0^{ii} = 0, "between two different atom sites")
                        const bool dg = (L == Lp);
                        for (int a = 0; a < nrep; ++a) {
                            const size_t item = (size_t)b + (size_t)a * rep_stride;
                            const c128* ti = tinv + (item * n_sites + si) * nspin * nt;
                            c128* cp = colp + (size_t)a * rep_elems;
                            if (!canted) {
                                cp[rowb] = (dg && !kbad) ? ti[lL] : zero;
                            } else {
                                const double* mv = moment + (item * n_sites + si) * 3;
                                const c128 ta = kbad ? zero : ti[lL], tb = kbad ? zero : ti[nt + lL];
                                const c128 hsum = cscale(0.5, cadd(ta, tb)), hdif = cscale(0.5, csub(ta, tb));
                                cp[rowb] = dg ? cadd(hsum, cscale(mv[2], hdif)) : zero;                         // (up, up)
                                cp[rowb + kmax] = dg ? cmul(hdif, cmake(mv[0], mv[1])) : zero;                  // (down, up): ex + i ey
                                cp[rowb + n * kmax] = dg ? cmul(hdif, cmake(mv[0], -mv[1])) : zero;             // (up, down): ex - i ey
                                cp[rowb + n * kmax + kmax] = dg ? csub(hsum, cscale(mv[2], hdif)) : zero;       // (down, down)
                            }
                        }
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------- host launchers

static size_t al256(size_t x) { return (x + 255) / 256 * 256; }

size_t gaunt_table_bytes(int lmax) {
    size_t kmax = (size_t)(lmax + 1) * (lmax + 1), nt = lmax + 1;
    size_t e = kmax * kmax * nt, S = (size_t)(2 * lmax + 1) * (2 * lmax + 1);
    return al256(e * sizeof(c128)) + al256(e * sizeof(int)) + al256(3 * S * sizeof(double));
}

int launch_tinv(const c128* delta, const int* species, const c128* z, int lmax, int n_sites, int nspin, int n_species, int batch,
                c128* tinv, c128* kappa, int* info, cudaStream_t st) {
    long long total = (long long)batch * n_sites * nspin * (lmax + 1);
    if (total < batch) total = batch;
    int thr = 256; long long blocks = (total + thr - 1) / thr;
    k_tinv<<<(unsigned)blocks, thr, 0, st>>>(delta, species, z, lmax, n_sites, nspin, n_species, batch, tinv, kappa, info);
    LSMS_LAUNCH_CHECK();
    return 0;
}

// n_rep > 1: de-duplicated assembly -- `batch` then counts the DISTINCT (geometry, kappa) items (the energies); item
// e + a*batch, a < n_rep, shares the geometry and kappa of item e and differs in tinv / moments only.
int init_attrs_assemble() {
    const int smem = 56 * 1024;
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_assemble<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_assemble<5, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_assemble<9, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_assemble<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_assemble<5, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_assemble<9, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    return 0;
}

int launch_assemble(const c128* tinv, const double* site_pos, const double* moment, const c128* kappa, int lmax,
                    int n_sites, int canted, int batch, int n_rep, c128* M, int* info, void* ws, cudaStream_t st) {
    size_t kmax = (size_t)(lmax + 1) * (lmax + 1), nt = lmax + 1, e = kmax * kmax * nt;
    const int l2 = 2 * lmax, nl2 = (l2 + 1) * (l2 + 1);
    c128* coef = (c128*)ws;
    int* idx = (int*)((char*)ws + al256(e * sizeof(c128)));
    double* leg = (double*)((char*)ws + al256(e * sizeof(c128)) + al256(e * sizeof(int)));
    k_gaunt_table<<<(unsigned)((e + 127) / 128) + 1, 128, 0, st>>>(lmax, coef, idx, leg);
    LSMS_LAUNCH_CHECK();
    // row-site chunks: per-R tables of a chunk fit in ~52 KB: four CTAs (32 warps) per SM hide the gather and
    // table latencies better than two with bigger chunks (measured on workload P: 3.7 ms vs 4.8 ms)
    int maxchunk = (int)((52 * 1024) / ((size_t)nl2 * sizeof(c128)));
    if (maxchunk < 1) maxchunk = 1;
    const int nchunks = (n_sites + maxchunk - 1) / maxchunk;
    const int chunk = (n_sites + nchunks - 1) / nchunks;      // balanced chunks
    const size_t smem = (size_t)chunk * nl2 * sizeof(c128);
    const size_t k = kmax * (canted ? 2 : 1), n = (size_t)n_sites * k;
    auto run = [&](auto kern) -> int {
        for (int b0 = 0; b0 < batch; b0 += 65535) {
            int nb = batch - b0 < 65535 ? batch - b0 : 65535;
            dim3 grid(n_sites, nb);
            kern<<<grid, ASM_THREADS, smem, st>>>(tinv + (size_t)b0 * n_sites * (canted ? 2 : 1) * nt,
                                                  site_pos + (size_t)b0 * n_sites * 3,
                                                  moment ? moment + (size_t)b0 * n_sites * 3 : nullptr, kappa + b0, coef, idx, leg,
                                                  lmax, n_sites, canted, chunk, n_rep, batch, M + (size_t)b0 * n * n, info + b0);
            LSMS_LAUNCH_CHECK();
        }
        return 0;
    };
    if (n_rep > 1) {
        if (lmax <= 3) return run(k_assemble<4, true>);
        if (lmax == 4) return run(k_assemble<5, true>);
        return run(k_assemble<9, true>);
    }
    if (lmax <= 3) return run(k_assemble<4, false>);
    if (lmax == 4) return run(k_assemble<5, false>);
    return run(k_assemble<9, false>);
}

}  // namespace lsms
