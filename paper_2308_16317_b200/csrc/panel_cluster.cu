// panel_cluster.cu -- K2 for tall panels of SMALL batches: one thread-block CLUSTER per matrix
// ("lets large ones span the whole chip"; PAPER.md:92 LU; pivot rule: reading A14).
//
// With one CTA per matrix (panel.cu) a batch of 12 rank-12450 matrices keeps 12 of the 148 SMs busy during the
// panel factorisation, and each CTA's rows-per-thread count forces 1-column sub-panels.  Here the rows of a panel
// are dealt round-robin to the CL CTAs of a cluster (CL = 2, 4 or 8; global thread g = rank*THREADS + tid owns
// rows c0 + g + r*CL*THREADS), so the sub-panel stays 4 columns wide and CL times as many SMs pull the panel
// through their load/store units.  Same algorithm and arithmetic as k_panel_reg; what crosses CTAs goes through
// distributed shared memory, every CTA keeping a full copy of the small shared state:
//   * column step: each warp finds its arg-max candidate (two redux.sync on a 64-bit key, as in panel_body.cuh) and
//     writes the candidate's ROW, the reciprocal of its would-be pivot and the key into slot [rank][warp] of EVERY
//     CTA; the owner of row j writes that row into every CTA; ONE cluster barrier; then every thread reduces the
//     CL*NW keys itself (same result everywhere) and has the pivot row in its own shared memory;
//   * L11, the rows of U: written by their owner into every CTA's copy;
//   * the interchanges of the outer panel's other columns and the final w x w solve are done by rank 0.
// Cluster barriers (arrive.release / wait.acquire, which also order the global-memory traffic between the CTAs of the
// cluster): one per column step, three more per sub-panel.
#include "common.cuh"
#include "internal.h"
#include "panel_body.cuh"

namespace lsms {

constexpr int PC_MAXW = 16;       // inner panel width limit
constexpr int PC_MAXOUT = 128;    // outer panel width limit
constexpr int PC_MAXCL = 8;       // portable cluster size limit

__device__ __forceinline__ uint32_t pc_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t pc_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t pc_nranks() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void pc_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared variable in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t pc_map(const void* p, uint32_t rank) {
    uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(pc_smem_u32(p)), "r"(rank)); return r;
}
__device__ __forceinline__ void pc_st_c128(uint32_t addr, c128 v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void pc_st_u64(uint32_t addr, unsigned long long v) { asm volatile("st.shared::cluster.u64 [%0], %1;" ::"r"(addr), "l"(v) : "memory"); }
__device__ __forceinline__ void pc_st_f64(uint32_t addr, double v) { asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory"); }
__device__ __forceinline__ void pc_st_s32(uint32_t addr, int v) { asm volatile("st.shared::cluster.s32 [%0], %1;" ::"r"(addr), "r"(v) : "memory"); }
// store v into the copy of *p held by every CTA of the cluster (including this one)
__device__ __forceinline__ void pc_bcast_c128(c128* p, c128 v, uint32_t ncl) { for (uint32_t k = 0; k < ncl; ++k) pc_st_c128(pc_map(p, k), v); }

template <int THREADS, int R, int S, int DEPTH>
__global__ void __launch_bounds__(THREADS, (THREADS <= 256) ? 2 : 1)
k_panel_clu(c128* __restrict__ base, size_t stride, int n, int J, int Wout, int c0, int w, int ne,
            int* __restrict__ piv, int* __restrict__ info) {
    constexpr int NW = THREADS / 32;
    static_assert(PC_MAXCL * R * THREADS <= 65536 && PC_MAXCL * NW <= 128,
                  "arg-max key: 16 bits for the row offset within the panel (65535 - offset), 7 for the (CTA, warp) slot");
    extern __shared__ __align__(16) unsigned char pc_stage[];
    c128* stage = reinterpret_cast<c128*>(pc_stage);
    const uint32_t rank = pc_rank(), ncl = pc_nranks();
    const int item = blockIdx.x / ncl;
    c128* A = base + (size_t)item * stride;
    int* pv = piv + (size_t)item * n;
    // column-step exchange, double-buffered by the parity of the column: per (CTA, warp) the candidate's row (S entries),
    // the reciprocal of its would-be pivot and the arg-max key; the row that stands at the pivot position
    __shared__ c128 cand[2][PC_MAXCL * NW][S + 2];
    __shared__ c128 jrow[2][S];
    __shared__ c128 L11[S * S];                 // L11[i*S + q] = multiplier of row cs+i, column cs+q (q < i)
    __shared__ c128 Us[S * PC_MAXW];            // Us[q*PC_MAXW + c] = U(cs+q, cs+sw+c)
    __shared__ int spiv[S], canon[S];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int TT = THREADS * (int)ncl;          // threads per matrix
    const int g0 = (int)rank * THREADS + tid;   // global thread index inside the cluster
    const int ncand = NW * (int)ncl;
    const c128 zero = cmake(0.0, 0.0);

    // every CTA of the cluster must be running before its shared memory is written from another CTA
    pc_sync();
    for (int s0 = 0; s0 < w; s0 += S) {
        const int cs = c0 + s0, sw = min(S, w - s0);
        // ---- 1: sub-panel -> registers
        c128 v[R][S];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int row = c0 + g0 + r * TT;
#pragma unroll
            for (int q = 0; q < S; ++q) v[r][q] = (row < n && q < sw) ? A[row + (size_t)(cs + q) * n] : zero;
        }
        // ---- 2: column steps, one cluster barrier each.  Arg-max key of a row: the bits of |re|+|im| with the low 23
        // mantissa bits replaced by (65535 - (row - c0), candidate slot): one unsigned 64-bit maximum picks the largest
        // magnitude and, among (nearly) equal ones, the lowest row; 0 = not eligible.
        int piv_reg[S];
#pragma unroll
        for (int q = 0; q < S; ++q) {
            piv_reg[q] = cs + q;
            if (q < sw) {
                const int j = cs + q, par = q & 1;
                const int myslot = (int)rank * NW + warp;
                // local best row by magnitude (ascending rows, strict >: the lowest row among equal ones), then ONE key
                double ba = -1.0; int rb = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int row = c0 + g0 + r * TT;
                    const double a = cabs1(v[r][q]);
                    if (row >= j && row < ne && (a > ba || a != a)) { ba = a; rb = r; }   // a NaN entry is taken, kept and flagged
                }
                unsigned long long key = 0ull;
                if (ba >= 0.0 || ba != ba)
                    key = ((unsigned long long)__double_as_longlong(ba) & ~0x7FFFFFull) |
                          ((unsigned long long)(65535 - (g0 + rb * TT)) << 7) | (unsigned long long)myslot;
                c128 vq = v[0][q];
#pragma unroll
                for (int r = 1; r < R; ++r) if (r == rb) vq = v[r][q];
                const c128 rinv = crecip_fast(vq);
                const uint32_t khi = (uint32_t)(key >> 32), klo = (uint32_t)key;
                const uint32_t mhi = __reduce_max_sync(0xffffffffu, khi);
                const uint32_t mlo = __reduce_max_sync(0xffffffffu, (khi == mhi) ? klo : 0u);
                if (key != 0ull && khi == mhi && klo == mlo) {
#pragma unroll 1
                    for (uint32_t kc = 0; kc < ncl; ++kc) {
                        const uint32_t dst = pc_map(&cand[par][myslot][0], kc);
#pragma unroll
                        for (int r = 0; r < R; ++r) if (r == rb) {
#pragma unroll
                            for (int t = 0; t < S; ++t) pc_st_c128(dst + t * (uint32_t)sizeof(c128), v[r][t]);
                        }
                        pc_st_c128(dst + S * (uint32_t)sizeof(c128), rinv);
                    }
                }
                if (lane < (int)ncl)
                    pc_st_u64(pc_map(&cand[par][myslot][S + 1], lane), ((unsigned long long)mhi << 32) | mlo);
                const int gj = j - c0;                      // row j belongs to cluster thread j - c0 (< 16 <= TT), its first row
                if (g0 == gj) {
#pragma unroll
                    for (int t = 0; t < S; ++t) pc_bcast_c128(&jrow[par][t], v[0][t], ncl);
                }
                pc_sync();
                // winner among the CL*NW candidates: every lane takes the slots lane, lane+32, ..., two more redux.sync
                unsigned long long ck = 0ull;
                for (int e = lane; e < ncand; e += 32) {
                    const unsigned long long ok = reinterpret_cast<const unsigned long long*>(&cand[par][e][S + 1])[0];
                    ck = ok > ck ? ok : ck;
                }
                const uint32_t chi = (uint32_t)(ck >> 32), clo = (uint32_t)ck;
                const uint32_t whi = __reduce_max_sync(0xffffffffu, chi);
                const uint32_t wlo = __reduce_max_sync(0xffffffffu, (chi == whi) ? clo : 0u);
                const unsigned long long wkey = ((unsigned long long)whi << 32) | wlo;
                const int wsel = (int)(wkey & 127ull);
                const bool bad = (wkey >> 23) == 0ull || (uint32_t)(wkey >> 52) >= 0x7FFu;     // zero, NaN or Inf pivot
                const int p = bad ? j : c0 + 65535 - (int)((wkey >> 7) & 0xFFFFull);
                piv_reg[q] = bad ? -1 - j : p;
                if (!bad) {
                    c128 prow[S];
#pragma unroll
                    for (int t = 0; t < S; ++t) prow[t] = cand[par][wsel][t];
                    const c128 rp = cand[par][wsel][S];
                    const int gp = (p - c0) % TT, rp_ = (p - c0) / TT;
                    if (p != j) {
                        if (g0 == gp) {
#pragma unroll
                            for (int r = 0; r < R; ++r) if (r == rp_) {
#pragma unroll
                                for (int t = 0; t < S; ++t) v[r][t] = jrow[par][t];
                            }
                        }
                        if (g0 == gj) {
#pragma unroll
                            for (int t = 0; t < S; ++t) v[0][t] = prow[t];
                        }
                    }
                    // ---- scale column j and rank-1 update of the sub-panel's remaining columns
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const int row = c0 + g0 + r * TT;
                        if (row > j && row < n) {
                            const c128 l = cmul(v[r][q], rp);
                            v[r][q] = l;
#pragma unroll
                            for (int t = q + 1; t < S; ++t) if (t < sw) cfms(v[r][t], l, prow[t]);
                        }
                    }
                }
            }
        }
        // ---- 3: store the sub-panel (rows above cs hold finished U entries and are unchanged); L11 to every CTA
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int row = c0 + g0 + r * TT;
            if (row >= cs && row < n) {
#pragma unroll
                for (int q = 0; q < S; ++q) if (q < sw) A[row + (size_t)(cs + q) * n] = v[r][q];
                if (row < cs + sw) {
#pragma unroll
                    for (int q = 0; q < S; ++q) pc_bcast_c128(&L11[(row - cs) * S + q], v[r][q], ncl);
                }
            }
        }
        if (tid == 0) {
#pragma unroll
            for (int q = 0; q < S; ++q) {
                if (q < sw) {
                    const int pq = piv_reg[q] < 0 ? -1 - piv_reg[q] : piv_reg[q];
                    spiv[q] = pq;
                    if (rank == 0) { pv[cs + q] = pq; if (piv_reg[q] < 0) atomicCAS(&info[item], 0, cs + q + 1); }
                }
            }
            // canon[i] = first step whose pivot row equals that of step i (rows below the sub-panel only)
            for (int i = 0; i < sw; ++i) {
                int c = -1;
                if (spiv[i] >= cs + sw) { c = i; for (int t = 0; t < i; ++t) if (spiv[t] == spiv[i]) { c = t; break; } }
                canon[i] = c;
            }
        }
        pc_sync();           // sub-panel stores (global) and L11 (shared) visible to the whole cluster
        // ---- 4 (rank 0): the other columns of the outer panel: interchanges (+ S x S solve for the inner panel's right part)
        const int nright = (c0 + w) - (cs + sw);          // inner-panel columns still to be updated
        if (rank == 0 && tid < Wout) {
            const int cu = J + tid;
            if (cu < cs || cu >= cs + sw) {
                c128* col = A + (size_t)cu * n;
                c128 x[S], y[S];
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    x[i] = (i < sw) ? col[cs + i] : zero;
                    y[i] = (i < sw && canon[i] == i) ? col[spiv[i]] : zero;
                }
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    if (i < sw) {
                        const int p = spiv[i];
                        if (p != cs + i) {
                            const int k = (p < cs + sw) ? (p - cs) : canon[i];
                            const bool top = p < cs + sw;
                            const c128 xi = x[i];
                            c128 other = xi;
#pragma unroll
                            for (int t = 0; t < S; ++t) if (t == k) other = top ? x[t] : y[t];
#pragma unroll
                            for (int t = 0; t < S; ++t) if (t == k) { if (top) x[t] = xi; else y[t] = xi; }
                            x[i] = other;
                        }
                    }
                }
                const bool right = cu >= cs + sw && cu < c0 + w;
                if (right) {
#pragma unroll
                    for (int jq = 0; jq < S; ++jq)
#pragma unroll
                        for (int i = jq + 1; i < S; ++i)
                            if (i < sw) cfms(x[i], L11[i * S + jq], x[jq]);
#pragma unroll
                    for (int i = 0; i < S; ++i) if (i < sw) pc_bcast_c128(&Us[i * PC_MAXW + (cu - cs - sw)], x[i], ncl);
                }
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    if (i < sw) {
                        col[cs + i] = x[i];
                        if (canon[i] == i) col[spiv[i]] = y[i];
                    }
                }
            }
        }
        pc_sync();           // interchanged columns (global) and the rows of U (shared) visible to the whole cluster
        // ---- 5: rank-sw update of the inner panel's remaining columns (rows below the sub-panel): the columns stream
        // through shared memory with per-thread asynchronous copies, DEPTH columns ahead (as in panel_body.cuh)
        if (nright > 0) {
            auto issue = [&](int c) {
                if (c < nright) {
                    c128* dst = stage + (size_t)(c % DEPTH) * (R * THREADS) + tid;
                    const c128* src = A + (size_t)(cs + sw + c) * n + c0 + g0;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const int row = c0 + g0 + r * TT;
                        if (row >= cs + sw && row < n) cp_async16(dst + r * THREADS, src + (size_t)r * TT);
                    }
                }
                cp_async_commit();
            };
            for (int d = 0; d < DEPTH; ++d) issue(d);
            for (int c = 0; c < nright; ++c) {
                cp_async_wait<DEPTH - 1>();
                const c128* src = stage + (size_t)(c % DEPTH) * (R * THREADS) + tid;
                c128 u[S];
#pragma unroll
                for (int q = 0; q < S; ++q) u[q] = (q < sw) ? Us[q * PC_MAXW + c] : zero;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int row = c0 + g0 + r * TT;
                    if (row >= cs + sw && row < n) {
                        c128 x = src[r * THREADS];
#pragma unroll
                        for (int q = 0; q < S; ++q) if (q < sw) cfms(x, v[r][q], u[q]);
                        A[row + (size_t)(cs + sw + c) * n] = x;
                    }
                }
                issue(c + DEPTH);
            }
            cp_async_wait<0>();
        }
        pc_sync();           // updated columns visible before the next sub-panel is loaded by other owners' neighbours
    }
    // ---- 6 (rank 0): U12 of the outer panel's columns to the RIGHT of this inner panel: the w x w unit-lower solve
    const int nr = (J + Wout) - (c0 + w);
    if (nr > 0 && rank == 0) {
        __shared__ c128 Lw[PC_MAXW * PC_MAXW];
        for (int e = tid; e < w * w; e += THREADS) { const int r = e % w, c = e / w; Lw[r + PC_MAXW * c] = A[(c0 + r) + (size_t)(c0 + c) * n]; }
        __syncthreads();
        if (tid < nr) {
            c128* col = A + (size_t)(c0 + w + tid) * n + c0;
            c128 x[PC_MAXW];
#pragma unroll
            for (int i = 0; i < PC_MAXW; ++i) x[i] = (i < w) ? col[i] : zero;
#pragma unroll
            for (int jq = 0; jq < PC_MAXW; ++jq)
#pragma unroll
                for (int i = jq + 1; i < PC_MAXW; ++i)
                    if (i < w) cfms(x[i], Lw[i + PC_MAXW * jq], x[jq]);
#pragma unroll
            for (int i = 0; i < PC_MAXW; ++i) if (i < w) col[i] = x[i];
        }
    }
}

template <int THREADS, int R, int DEPTH> constexpr size_t pc_stage_bytes() { return (size_t)DEPTH * R * THREADS * sizeof(c128); }

template <int THREADS, int R, int S, int DEPTH>
static int launch_clu(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                      int cl, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(batch * cl), 1, 1);
    cfg.blockDim = dim3(THREADS, 1, 1);
    cfg.dynamicSmemBytes = pc_stage_bytes<THREADS, R, DEPTH>();
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    LSMS_CUDA_OK(cudaLaunchKernelEx(&cfg, k_panel_clu<THREADS, R, S, DEPTH>, base, stride, n, J, Wout, c0, w, ne, piv, info));
    LSMS_LAUNCH_CHECK();
    return 0;
}

// (THREADS, R rows per thread, S sub-panel width, DEPTH columns in flight in step 5)
#define LSMS_PC_LIST(X) X(256, 1, 4, 4) X(256, 2, 4, 4) X(512, 2, 4, 4) X(512, 5, 4, 4) X(512, 10, 2, 2)

int init_attrs_panel_cluster() {
#define LSMS_PC_ATTR(T, R, S, D) \
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_panel_clu<T, R, S, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pc_stage_bytes<T, R, D>()));
    LSMS_PC_LIST(LSMS_PC_ATTR)
#undef LSMS_PC_ATTR
    return 0;
}

template <int THREADS, int R, int S, int DEPTH>
static int active_clu(int cl) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)cl, 1, 1); cfg.blockDim = dim3(THREADS, 1, 1); cfg.dynamicSmemBytes = pc_stage_bytes<THREADS, R, DEPTH>();
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cl; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    int nclu = 0;
    if (cudaOccupancyMaxActiveClusters(&nclu, k_panel_clu<THREADS, R, S, DEPTH>, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return nclu;
}

// the minimum over the instances: a panel walks through several of them as it gets shorter
int panel_cluster_max_active_clusters(int cl) {
    if (cl < 2 || cl > PC_MAXCL) return 0;
    int best = 1 << 30;
#define LSMS_PC_OCC(T, R, S, D) { const int a = active_clu<T, R, S, D>(cl); if (a < best) best = a; }
    LSMS_PC_LIST(LSMS_PC_OCC)
#undef LSMS_PC_OCC
    return best;
}

// cl = CTAs per matrix (2, 4 or 8); rows per CTA = ceil((n - c0) / cl) picks the instance
int launch_panel_cluster(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                         int cl, cudaStream_t st) {
    if (w < 1 || w > PC_MAXW || Wout > PC_MAXOUT || cl < 2 || cl > PC_MAXCL) return -1;
    const int m = (n - c0 + cl - 1) / cl;
#define LSMS_PC(T, R, S, D) return launch_clu<T, R, S, D>(base, stride, n, J, Wout, c0, w, ne, batch, piv, info, cl, st)
    if (m <= 256) LSMS_PC(256, 1, 4, 4);
    if (m <= 512) LSMS_PC(256, 2, 4, 4);
    if (m <= 1024) LSMS_PC(512, 2, 4, 4);
    if (m <= 2560) LSMS_PC(512, 5, 4, 4);
    if (m <= 5120) LSMS_PC(512, 10, 2, 2);
#undef LSMS_PC
    return -1;
}

}  // namespace lsms
