// kernels.cu -- __global__ wrappers and launchers (see kernels.cuh for the per-thread code).  sm_100a only.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>

#include "kernels.cuh"
#include "kernels.h"

namespace gv {

// ---- parameter expansion: (cos(theta/2), sin(theta/2)) in fp64, stored in working precision ----
// Second output for the specialised gate kernels (jit.cpp): R_y(theta) = c [[1,-t],[t,1]] with t = s/c when |c| >= |s|
// (form 0), else s [[t,-1],[1,t]] with t = c/s (form 1); {t, scale = c or s, form, 0} per parameter (Eq. 7).
template <typename T> struct alignas(4 * sizeof(T)) ry4 { T t, sc, form, pad; };
template <typename T>
__global__ void expand_params_kernel(const double *__restrict__ params, cx<T> *__restrict__ cs, ry4<T> *__restrict__ ry, uint64_t count)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    double s, c;
    sincos(0.5 * params[i], &s, &c);
    cs[i] = cx<T>{(T)c, (T)s};
    if (ry) {
        const bool f0 = fabs(c) >= fabs(s);
        ry[i] = ry4<T>{(T)(f0 ? s / c : c / s), (T)(f0 ? c : s), f0 ? T(0) : T(1), T(0)};
    }
}

// ---- rows of a parameter-shift set (Eq. 13): row r = theta with +/- pi/2 on parameter code[r] >> 1 ----
__global__ void __launch_bounds__(256) shift_rows_kernel(const double *__restrict__ theta, const int32_t *__restrict__ code,
                                                         double *__restrict__ rows, int P)
{
    const int p = code[blockIdx.x] >> 1;
    const double d = (code[blockIdx.x] & 1) ? -1.57079632679489661923 : 1.57079632679489661923;
    for (int i = threadIdx.x; i < P; i += blockDim.x) rows[(size_t)blockIdx.x * P + i] = theta[i] + (i == p ? d : 0.0);
}

int launch_shift_rows(const double *theta, const int32_t *code, double *rows, int P, int n_rows, void *stream, uint64_t *launches)
{
    if (n_rows <= 0) return 0;
    shift_rows_kernel<<<n_rows, 256, 0, (cudaStream_t)stream>>>(theta, code, rows, P);
    ++*launches;
    return (int)cudaGetLastError();
}

// ---- product-state prefix, write-only --------------------------------------------------------------
// psi[y] = sign(y) * prod_q f_q[x_q],  x = A^-1 y  (A = the prefix's CNOT run, linear over GF(2); sign = its CZ run),
// f_q = (rotations of qubit q)|0>.  The product comes from tables over 7-qubit groups; A^-1 y is split into the
// thread's part, the vector's part and the lane-in-vector part (linearity), so nothing per amplitude depends on
// the number of CNOTs.  Each thread block writes 2^kk contiguous amplitudes with 16-byte stores.
__device__ __forceinline__ uint64_t prefix_ainv(const PrefixDev &pd, uint64_t y)
{
    for (int i = pd.n_cx - 1; i >= 0; --i) y ^= ((y >> pd.cx_c[i]) & 1ull) << pd.cx_t[i];
    return y;
}

// The x bits that differ among the 2^kk amplitudes of one thread block (pd.vary, m = pd.n_vary of them) are numbered
// 0 .. m-1 ("compact index"); A^-1 is linear, so the compact index of an amplitude is the XOR of the images pd.cimg[b] of
// the set bits b of its offset inside the thread block.  The product over those m qubits comes from NTAB tables of 256
// entries (8 compact bits each) rebuilt by every thread block with its own x folded in; the product over the other
// qubits is one constant per thread block, folded into table 0.  Per amplitude: NTAB lookups, NTAB - 1 multiplications.
template <typename T, int NTAB>
__global__ void __launch_bounds__(256, 4)
init_product_kernel(const __grid_constant__ PrefixDev pd, cx<T> *states, uint64_t stride, const cx<T> *cs_table, int P)
{
    __shared__ cx<T> f[40][2];
    __shared__ cx<T> tab[NTAB][256];
    __shared__ uint64_t cxi[64];
    __shared__ cx<T> pconst;
    constexpr uint32_t V = 16 / sizeof(cx<T>);
    constexpr int LV = V == 2 ? 1 : 0;
    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    const cx<T> *cs = cs_table + (uint64_t)blockIdx.y * P;
    cx<T> *state = states + (uint64_t)blockIdx.y * stride;
    const int n = pd.n;
    if ((int)tid < n) {   // f_q = U_m ... U_1 |0>, Eq. 7
        cx<T> a{T(1), T(0)}, b{T(0), T(0)};
        for (int r = pd.rot_begin[tid]; r < pd.rot_begin[tid + 1]; ++r) {
            const cx<T> v = cs[pd.rot_param[r]];   // (cos, sin) of theta / 2
            if (pd.rot_kind[r] == 0) {
                const cx<T> a2{v.x * a.x - v.y * b.x, v.x * a.y - v.y * b.y}, b2{v.y * a.x + v.x * b.x, v.y * a.y + v.x * b.y};
                a = a2; b = b2;
            } else { a = cmul(a, cx<T>{v.x, -v.y}); b = cmul(b, v); }
        }
        f[tid][0] = a; f[tid][1] = b;
    }
    const uint32_t nvec = (1u << pd.kk) / V / nthr;   // vectors per thread (<= 64)
    const int tbits = 31 - __clz(nthr);                // offset bits [LV, LV + tbits) belong to the thread, the ones above to the vector number
    if (tid < nvec) {
        uint64_t c = 0;
        for (int b = 0; (1u << b) < nvec; ++b) if ((tid >> b) & 1u) c ^= pd.cimg[LV + tbits + b];
        cxi[tid] = c;
    }
    const uint64_t xcta = prefix_ainv(pd, (uint64_t)blockIdx.x << pd.kk);   // x of the thread block's first amplitude
    __syncthreads();
    if (tid < 32) {   // product over the qubits whose x bit is the same for the whole thread block
        cx<T> p{T(1), T(0)};
        for (int q = (int)tid; q < n; q += 32)
            if (!((pd.vary >> q) & 1ull)) p = cmul(p, f[q][(xcta >> q) & 1ull]);
        for (int o = 16; o > 0; o >>= 1) {
            cx<T> r;
            r.x = __shfl_xor_sync(0xffffffffu, p.x, o); r.y = __shfl_xor_sync(0xffffffffu, p.y, o);
            p = cmul(p, r);
        }
        if (tid == 0) pconst = p;
    }
    __syncthreads();
    for (uint32_t e = tid; e < (uint32_t)NTAB * 256u; e += nthr) {
        const uint32_t g = e >> 8, v = e & 255u;
        cx<T> p = g == 0 ? pconst : cx<T>{T(1), T(0)};
        for (int j = 0; j < 8 && (int)(8 * g) + j < pd.n_vary; ++j) {
            const int q = pd.vq[8 * g + j];
            p = cmul(p, f[q][((xcta >> q) ^ (uint64_t)(v >> j)) & 1ull]);
        }
        tab[g][v] = p;
    }
    uint64_t cthr = 0;
    for (int b = 0; b < tbits; ++b) if ((tid >> b) & 1u) cthr ^= pd.cimg[LV + b];
    const uint64_t ce1 = V > 1 ? pd.cimg[0] : 0ull;
    const bool e_low = (ce1 >> 8) == 0ull;   // the lane-in-vector bit moves table 0 only: the other factors are shared by the vector
    const uint64_t ybase = ((uint64_t)blockIdx.x << pd.kk) | (uint64_t)(tid * V);
    __syncthreads();
    for (uint32_t i = 0; i < nvec; ++i) {
        vec16<T> out;
        const uint64_t c0 = cthr ^ cxi[i];
        cx<T> rest{T(1), T(0)};
        if (NTAB > 1 && e_low) {
            rest = tab[1][(c0 >> 8) & 255ull];
#pragma unroll
            for (int g = 2; g < NTAB; ++g) rest = cmul(rest, tab[g][(c0 >> (8 * g)) & 255ull]);
        }
#pragma unroll
        for (uint32_t e = 0; e < V; ++e) {
            const uint64_t y = ybase | ((uint64_t)i * nthr * V) | e;
            const uint64_t c = c0 ^ (e ? ce1 : 0ull);
            cx<T> p = tab[0][c & 255ull];
            if (NTAB > 1) {
                if (e_low) p = cmul(p, rest);
                else {
#pragma unroll
                    for (int g = 1; g < NTAB; ++g) p = cmul(p, tab[g][(c >> (8 * g)) & 255ull]);
                }
            }
            int par = 0;
            for (int cz = 0; cz < pd.n_cz; ++cz) par += __popcll(y & (y >> pd.cz_d[cz]) & pd.cz_m[cz]);
            out.v[e] = (par & 1) ? cneg(p) : p;
        }
        *reinterpret_cast<vec16<T> *>(state + (ybase | ((uint64_t)i * nthr * V))) = out;
    }
}

// ---- fused gate block: one HBM round trip, all stages of the block in shared memory ---------
template <typename T, int R, int MAXT>
__global__ void __launch_bounds__(MAXT, (MAXT <= 256 || R <= 4 ? 2 : 1))
gate_block_kernel(const DevArrays da, const __grid_constant__ DBlock blk, cx<T> *states, uint64_t stride,
                  const cx<T> *cs_table, int P)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const DBlock *sb = &blk;   // kernel parameter (constant bank): no load latency before the tile loads start
    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    ProgView<T> pv;
    cx<T> *tile = reinterpret_cast<cx<T> *>(smem + HDR_BYTES);   // fixed offset: LDS/STS take it as an immediate
    pv.bind(smem + HDR_BYTES + ((size_t)sizeof(cx<T>) << sb->k), *sb);
    const uint32_t b = blockIdx.y;
    cx<T> *state = states + (uint64_t)b * stride;
    const int k = sb->k, n_runs = sb->n_runs;
    const uint64_t xbase = tile_base(blockIdx.x, sb->runs, n_runs);
    const bool zero = sb->source_zero != 0;
    constexpr int NLD = (1 << R) / (16 / (int)sizeof(cx<T>));   // 16-byte vectors per thread
    const uint64_t *hi = sb->hi;
    if (zero && xbase != 0) {   // |0...0> has no weight in this tile and gates act inside tiles: stays zero
        tile_zero_store<T>(state, xbase, sb->runs, n_runs, k, tid, nthr);
        return;
    }
    // tile loads first (they need nothing but the kernel parameters) so that the program slice is fetched under them
    vec16<T> ld[NLD];
    const uint64_t x0 = xbase | scatter_runs(tid * (16 / (uint32_t)sizeof(cx<T>)), sb->runs, n_runs);
    if (!zero) {
#pragma unroll
        for (int i = 0; i < NLD; ++i) ld[i] = *reinterpret_cast<const vec16<T> *>(state + (x0 | hi[i]));
    }
    gate_prologue<T>(pv, *sb, da, cs_table + (uint64_t)b * P, tid, nthr);
    if (zero) tile_init_zero_state<T>(tile, k, tid, nthr);
    __syncthreads();   // program slice visible; the tile loads are still in flight and the phase tables are built under them
    for (uint32_t item = tid; item < sb->n_segs * TPH_CONST; item += nthr)
        tph_build_entry<T, R>(pv, item, xbase, sb->runs, n_runs, k);
    for (uint32_t sgi = tid >> 5; sgi < sb->n_segs; sgi += nthr >> 5) {   // tile-constant factors: one warp per segment
        const DSeg &sg = pv.segs[sgi];
        cx<T> pr{T(1), T(0)};
        for (uint32_t t = sg.trz_begin + sg.n_xreg + (tid & 31u); t < sg.trz_end; t += 32u) pr = cmul(pr, tph_const_factor<T>(pv, t, xbase));
        for (int o = 16; o > 0; o >>= 1) {
            cx<T> other;
            other.x = __shfl_xor_sync(0xffffffffu, pr.x, o);
            other.y = __shfl_xor_sync(0xffffffffu, pr.y, o);
            pr = cmul(pr, other);
        }
        if ((tid & 31u) == 0) pv.tph[sgi * TPH_ENTRIES + TPH_CONST] = pr;
    }
    if (zero) {
        if (tid == 0) tile[0] = cx<T>{T(1), T(0)};
    } else if (sb->lead_cx) {
        if (sb->n_lead_cx) tile_commit_cx<T, NLD>(tile, ld, tid, xbase, sb->lead_cxs, sb->n_lead_cx, sb->hip_cx, sb->e1_cx);
        else {
            const DStage *s0 = da.stages + sb->stage_off;
            tile_commit_cx<T, NLD>(tile, ld, tid, xbase, da.cxs + sb->cx_off + s0->cx_begin,
                                   (uint32_t)(s0->cx_end - s0->cx_begin), sb->hip_cx, sb->e1_cx);
        }
    } else tile_commit<T, NLD>(tile, ld, tid, sb->hip);
    __syncthreads();   // tile and phase tables visible
    const int ns = sb->n_stages;
    cx<T> amp[1 << R];
    uint32_t po[R], pj2 = 0;
    for (int s = (int)sb->lead_cx; s < ns; ++s) {
        if (gate_stage<T, R>(pv, pv.stages[s], (uint32_t)s, reinterpret_cast<unsigned char *>(tile), tid, xbase, amp, po, pj2)) {
            __syncthreads();   // reads done before the permuted writes
            gate_stage_store<T, R>(reinterpret_cast<unsigned char *>(tile), pj2, po, amp);
        }
        __syncthreads();
    }
    tile_store_u<T, NLD>(tile, state, x0, tid, hi, sb->hip);
}

constexpr uint32_t SGR_STRIDE = (uint32_t)((sizeof(DGroup) + 15) / 16 * 16);   // == sizeof(DGroup): shared-memory copy of a batch's groups

// ---- expectation pass: read-only sweep, diagonal table + every flip-mask group of the pass --
__device__ __forceinline__ double block_sum(double v, double *red)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) red[w] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0) for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += red[i];
    return s;   // valid on thread 0
}

template <typename T, typename TT, int L>
__global__ void __launch_bounds__(256, 2)
expect_pass_kernel(const DPass *passes, int pi, const DGroup *__restrict__ groups, const DTerm *__restrict__ terms,
                   const cx<T> *__restrict__ wstat, const uint32_t *__restrict__ gtabs, const DRs *__restrict__ rss,
                   const cx<T> *states, uint64_t stride, const TT *__restrict__ table,
                   double *partial, uint32_t slots_per_b, uint32_t slot_off, uint32_t nbatch)
{
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ double red[32];
    DPass *sp = reinterpret_cast<DPass *>(smem);
    const uint32_t tid = threadIdx.x, nthr = blockDim.x;   // nthr = 2^(k-1-L)
    {
        const uint32_t *src = reinterpret_cast<const uint32_t *>(passes + pi);
        uint32_t *dst = reinterpret_cast<uint32_t *>(sp);
        for (uint32_t i = tid; i < sizeof(DPass) / 4; i += nthr) dst[i] = src[i];
    }
    __syncthreads();
    constexpr int V = 16 / (int)sizeof(cx<T>);
    constexpr int NLD = (2 << L) / V;
    static_assert(sizeof(DPass) <= EXPECT_HDR_BYTES, "DPass must fit the shared-memory header");
    const uint64_t *hi = sp->hi;   // host-built vector offsets
    cx<T> *tab = reinterpret_cast<cx<T> *>(smem + EXPECT_HDR_BYTES);
    uint32_t *gts = reinterpret_cast<uint32_t *>(tab + EXPECT_TAB_CAP);
    DGroup *sgr = reinterpret_cast<DGroup *>(gts + GT_BATCH_MAX * GT_WORDS);
    cx<T> *tile = reinterpret_cast<cx<T> *>(reinterpret_cast<unsigned char *>(sgr) + GT_BATCH_MAX * SGR_STRIDE);
    // linear grid, batch fastest: the thread blocks that work on the same tile of different statevectors run together,
    // so the diagonal table, the static W tables and the lookup blocks they share are served from L2
    const uint32_t b = blockIdx.x % nbatch, tile_id = blockIdx.x / nbatch;
    const cx<T> *state = states + (uint64_t)b * stride;
    const int k = sp->k, n_runs = sp->n_runs;
    const uint64_t xbase = tile_base(tile_id, sp->runs, n_runs);
    double acc = expect_load_u<T, TT, NLD>(tile, state, table, sp->with_diag != 0, xbase, sp->runs, n_runs, tid, nthr, hi);
    __syncthreads();
    for (uint32_t bi = 0; bi < sp->n_batches; ++bi) {
        const uint32_t g = sp->batch[bi].g_first, ge = sp->batch[bi].g_last;
        {   // the batch's group descriptors, static W tables and lookup blocks: three contiguous global ranges copied by
            // ONE loop of independent 8-byte loads (a single round of L2 latency)
            struct alignas(8) u2 { uint32_t a, b; };
            const uint32_t ng = ge - g + 1;
            const uint32_t nd = ng * (uint32_t)(sizeof(DGroup) / 8), nt = sp->batch[bi].entries * (uint32_t)(sizeof(cx<T>) / 8),
                           nl = ng * (GT_WORDS / 2);
            const u2 *s_d = reinterpret_cast<const u2 *>(groups + g);
            const u2 *s_t = reinterpret_cast<const u2 *>(wstat + sp->batch[bi].wbase);
            const u2 *s_l = reinterpret_cast<const u2 *>(gtabs + (uint64_t)g * GT_WORDS);
            u2 *d_d = reinterpret_cast<u2 *>(sgr), *d_t = reinterpret_cast<u2 *>(tab), *d_l = reinterpret_cast<u2 *>(gts);
            for (uint32_t i = tid; i < nd + nt + nl; i += nthr) {
                if (i < nd) d_d[i] = s_d[i];
                else if (i < nd + nt) d_t[i - nd] = s_t[i - nd];
                else d_l[i - nd - nt] = s_l[i - nd - nt];
            }
        }
        __syncthreads();
        // tile-dependent terms (z bits outside the tile) on top: small tables one warp per group (different groups
        // concurrently), large tables with the whole block
        for (uint32_t gi = g + (tid >> 5); gi <= ge; gi += (nthr >> 5)) {
            const DGroup *pg = sgr + (gi - g);
            if (!(pg->hot >> 63) || pg->ubits > 6) continue;
            const uint32_t tb = pg->term_begin, de = pg->dyn_end, to = pg->tab_off, ne = 1u << pg->ubits;
            for (uint32_t u = tid & 31u; u < ne; u += 32u)
                tab[to + u] = group_table_entry<T>(tb, de, terms, xbase, u, tab[to + u]);
        }
        for (uint32_t gi = g; gi <= ge; ++gi) {
            const DGroup *pg = sgr + (gi - g);
            if (!(pg->hot >> 63) || pg->ubits <= 6) continue;
            const uint32_t tb = pg->term_begin, de = pg->dyn_end, to = pg->tab_off, ne = 1u << pg->ubits;
            for (uint32_t u = tid; u < ne; u += nthr)
                tab[to + u] = group_table_entry<T>(tb, de, terms, xbase, u, tab[to + u]);
        }
        __syncthreads();
        int cur_rs = -1;
        constexpr int RSR = (L + 1 <= DEV_MAX_R) ? L + 1 : 1;   // the planner makes register stages only when L + 1 <= DEV_MAX_R
        cx<T> ra[1 << RSR];   // register stage: 2^(L+1) amplitudes per thread
        uint64_t hot_next = sgr[0].hot;   // one group ahead: the shared-memory read overlaps the previous group's pairs
        for (uint32_t gi = g; gi <= ge; ++gi) {
            const DGroup *pg = sgr + (gi - g);
            const uint64_t hot = hot_next;
            if (gi < ge) hot_next = pg[1].hot;
            const uint32_t mode = (uint32_t)hot & 3u, tab_off = (uint32_t)(hot >> 24) & 0xFFFFFFu;
            if (mode == 1u) {
                const int rs_id = (int)((hot >> 8) & 0xFFFFu);
                if (rs_id != cur_rs) {
                    cur_rs = rs_id;
                    rs_load<T, RSR>(ra, rss[cur_rs], reinterpret_cast<const unsigned char *>(tile), tid);
                }
                acc += 2.0 * (double)RsDispatch<T, RSR, 1, (1 << RSR) - 1>::run((int)((hot >> 2) & 63u), ra, tab + tab_off);
            } else if (mode == 2u) {
                const DGroup dg = *pg;
                acc += group_accumulate<T>(dg, terms, tile, tab, xbase, k, tid, nthr);
            } else {
                acc += group_accumulate_lut<T, L>(gts + (gi - g) * GT_WORDS, pg->pm_bytes, tab_off,
                                                  reinterpret_cast<const unsigned char *>(tile), tab, tid);
            }
        }
        __syncthreads();
    }
    const double s = block_sum(acc, red);
    if (tid == 0) partial[(uint64_t)b * slots_per_b + slot_off + tile_id] = s;
}

// ---- second-stage deterministic reduction ------------------------------------------------------
// Large slot counts (one statevector of 2^32 amplitudes has 2^19 tiles per pass) are summed in two steps: slice c of a
// row is reduced into the first element of that slice, then the slice heads are summed.  Fixed order: deterministic.
__global__ void __launch_bounds__(256) reduce_slices_kernel(double *partial, uint32_t slots_per_b, uint32_t slice_len)
{
    __shared__ double red[32];
    double *p = partial + (uint64_t)blockIdx.y * slots_per_b + (uint64_t)blockIdx.x * slice_len;
    const uint32_t n = min(slice_len, slots_per_b - blockIdx.x * slice_len);
    double v = 0.0;
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) v += p[i];
    const double s = block_sum(v, red);   // contains the barrier that orders every read before the write below
    if (threadIdx.x == 0) p[0] = s;
}

__global__ void __launch_bounds__(256) reduce_kernel(const double *__restrict__ partial, uint32_t slots_per_b, uint32_t stride,
                                                     double *E)
{
    __shared__ double red[32];
    const double *p = partial + (uint64_t)blockIdx.x * slots_per_b;
    double v = 0.0;
    for (uint32_t i = threadIdx.x * stride; i < slots_per_b; i += blockDim.x * stride) v += p[i];
    const double s = block_sum(v, red);
    if (threadIdx.x == 0) E[blockIdx.x] = s;
}

// ---- read-out ("the bitstring with the highest probability") -------------------
// One read-only sweep: every thread keeps the best (|psi_x|^2, x) of its 16-byte vectors, ties to the lowest x; warp
// shuffles, one entry per block, then a single block picks the winner.  max / lowest-index are order independent, so
// the result does not depend on the grid.  |psi|^2 = re*re + im*im in the working precision, each operation rounded
// separately (no FMA contraction) so that the decision is reproducible outside the kernel.
struct ProbIdx { double p; uint64_t x; };
__device__ __forceinline__ float prob_of(cx<float> a) { return __fadd_rn(__fmul_rn(a.x, a.x), __fmul_rn(a.y, a.y)); }
__device__ __forceinline__ double prob_of(cx<double> a) { return __dadd_rn(__dmul_rn(a.x, a.x), __dmul_rn(a.y, a.y)); }
__device__ __forceinline__ void take_better(double &p, uint64_t &x, double q, uint64_t y)
{
    if (q > p || (q == p && y < x)) { p = q; x = y; }
}
__device__ __forceinline__ void block_best(double &p, uint64_t &x, ProbIdx *red)
{
    for (int o = 16; o > 0; o >>= 1) {
        const double q = __shfl_down_sync(0xffffffffu, p, o);
        const uint64_t y = __shfl_down_sync(0xffffffffu, x, o);
        take_better(p, x, q, y);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) red[w] = ProbIdx{p, x};
    __syncthreads();
    if (threadIdx.x == 0)
        for (int i = 1; i < (int)(blockDim.x >> 5); ++i) take_better(p, x, red[i].p, red[i].x);
}

template <typename T>
__global__ void __launch_bounds__(256, 8) argmax_partial_kernel(const cx<T> *__restrict__ state, uint64_t count, ProbIdx *out)
{
    __shared__ ProbIdx red[8];
    constexpr uint32_t V = 16 / (uint32_t)sizeof(cx<T>);
    constexpr int U = 4;   // independent 16-byte loads in flight per thread (8 resident blocks per SM: one wave of 148 x 8)
    double bp = -1.0;
    uint64_t bx = ~0ull;
    const uint64_t nvec = count / V, step = (uint64_t)gridDim.x * 256u;
    uint64_t i = (uint64_t)blockIdx.x * 256u + threadIdx.x;
    for (; i + (U - 1) * step < nvec; i += U * step) {
        vec16<T> v[U];
#pragma unroll
        for (int r = 0; r < U; ++r) v[r] = *reinterpret_cast<const vec16<T> *>(state + (i + r * step) * V);
#pragma unroll
        for (int r = 0; r < U; ++r)
#pragma unroll
            for (uint32_t j = 0; j < V; ++j) take_better(bp, bx, (double)prob_of(v[r].v[j]), (i + r * step) * V + j);
    }
    for (; i < nvec; i += step) {
        const vec16<T> v = *reinterpret_cast<const vec16<T> *>(state + i * V);
#pragma unroll
        for (uint32_t j = 0; j < V; ++j) take_better(bp, bx, (double)prob_of(v.v[j]), i * V + j);
    }
    if (count < V && blockIdx.x == 0 && threadIdx.x == 0)   // a one-amplitude register
        for (uint64_t x = 0; x < count; ++x) take_better(bp, bx, (double)prob_of(state[x]), x);
    block_best(bp, bx, red);
    if (threadIdx.x == 0) out[blockIdx.x] = ProbIdx{bp, bx};
}

__global__ void __launch_bounds__(256) argmax_final_kernel(const ProbIdx *__restrict__ part, uint32_t n_part, ProbIdx *out)
{
    __shared__ ProbIdx red[8];
    double bp = -1.0;
    uint64_t bx = ~0ull;
    for (uint32_t i = threadIdx.x; i < n_part; i += 256u) take_better(bp, bx, part[i].p, part[i].x);
    block_best(bp, bx, red);
    if (threadIdx.x == 0) *out = ProbIdx{bp, bx};
}

int launch_argmax(int prec, const void *state, uint64_t count, void *scratch, void *stream, uint64_t *launches)
{
    const uint64_t nvec = count / (prec == 0 ? 2 : 1);
    uint32_t grid = (uint32_t)std::min<uint64_t>(READOUT_BLOCKS, (nvec + 255) / 256);
    if (grid == 0) grid = 1;
    ProbIdx *part = reinterpret_cast<ProbIdx *>(scratch);   // [0] = result, [1 ..] = per-block entries
    if (prec == 0) argmax_partial_kernel<float><<<grid, 256, 0, (cudaStream_t)stream>>>((const cx<float> *)state, count, part + 1);
    else argmax_partial_kernel<double><<<grid, 256, 0, (cudaStream_t)stream>>>((const cx<double> *)state, count, part + 1);
    argmax_final_kernel<<<1, 256, 0, (cudaStream_t)stream>>>(part + 1, grid, part);
    *launches += 2;
    return (int)cudaGetLastError();
}

// ---- the same read-out for callers that may not allocate (gvqe_argmax_noalloc, include/gvqe.h) ----------------------
// The per-block entries live in a file-scope device array instead of a workspace: NOALLOC_SCRATCH_BYTES on every GPU that
// loads the library, until the process exits.  Every call on a device shares it and it keeps the last call's contents;
// nothing in it has to start at zero (the final kernel reads exactly the entries the first kernel of the same call
// wrote), but two calls that overlap on the GPU (different streams) race on it.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
void *g_noalloc_ptr[NOALLOC_MAX_DEVICES];     // device address of g_noalloc_scratch, per device ordinal
std::atomic<int> g_noalloc_state[NOALLOC_MAX_DEVICES];   // 0 = not looked up, 1 = ready
}  // namespace

// Device address of the scratch array on the CURRENT device.  In host code the name g_noalloc_scratch is only a handle
// for the runtime, not a device address: the address comes from cudaGetSymbolAddress, once per device.
static int noalloc_scratch_address(void **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return (int)cudaErrorInvalidDevice;
    if (g_noalloc_state[dev].load(std::memory_order_acquire) != 1) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess) return (int)e;
        if (!ptr) return (int)cudaErrorInvalidSymbol;
        g_noalloc_ptr[dev] = ptr;   // concurrent first calls store the same value
        g_noalloc_state[dev].store(1, std::memory_order_release);
    }
    *out = g_noalloc_ptr[dev];
    return 0;
}

int launch_argmax_noalloc(int prec, const void *state, uint64_t count, void *result, void *stream)
{
    void *scratch = nullptr;
    const int se = noalloc_scratch_address(&scratch);
    if (se) return se;
    const uint64_t nvec = count / (prec == 0 ? 2 : 1);
    uint32_t grid = (uint32_t)std::min<uint64_t>(READOUT_BLOCKS, (nvec + 255) / 256);   // as launch_argmax: same partition, same result
    if (grid == 0) grid = 1;
    static_assert((size_t)READOUT_BLOCKS * sizeof(ProbIdx) <= NOALLOC_SCRATCH_BYTES, "scratch array too small");
    ProbIdx *part = reinterpret_cast<ProbIdx *>(scratch);
    if (prec == 0) argmax_partial_kernel<float><<<grid, 256, 0, (cudaStream_t)stream>>>((const cx<float> *)state, count, part);
    else argmax_partial_kernel<double><<<grid, 256, 0, (cudaStream_t)stream>>>((const cx<double> *)state, count, part);
    argmax_final_kernel<<<1, 256, 0, (cudaStream_t)stream>>>(part, grid, reinterpret_cast<ProbIdx *>(result));
    return (int)cudaGetLastError();
}

// ---- shot sampling ("this state is sampled", 256: 8192 shots) ---------------------
// Inverse-CDF sampling from uniforms the caller supplies: x_s = the first x whose cumulative probability exceeds
// u_s * Z, Z = sum_x |psi_x|^2.  Three kernels: probability mass of every chunk of 2^SAMPLE_CHUNK_LOG2 amplitudes
// (fp64, fixed order), exclusive prefix over the chunks (one block, fixed order), then one warp per shot: binary
// search over the chunk prefixes and a 32-wide running scan inside the chunk.  Deterministic.
template <typename T>
__global__ void __launch_bounds__(256, 6) chunk_mass_kernel(const cx<T> *__restrict__ state, uint64_t count, uint32_t chunk_len,
                                                            double *__restrict__ mass, uint64_t n_chunks)
{
    // one warp per chunk (no block barrier): lane-local sums over 16-byte vectors, four loads in flight, then shuffles
    constexpr uint32_t V = 16 / (uint32_t)sizeof(cx<T>);
    const uint32_t lane = threadIdx.x & 31u;
    const uint64_t nwarps = (uint64_t)gridDim.x * 8u;
    for (uint64_t ci = (uint64_t)blockIdx.x * 8u + (threadIdx.x >> 5); ci < n_chunks; ci += nwarps) {
        const cx<T> *p = state + ci * chunk_len;
        const uint32_t len = (uint32_t)min((uint64_t)chunk_len, count - ci * chunk_len);
        double v = 0.0;
        if (len == chunk_len) {
            const uint32_t nv = chunk_len / V;   // a multiple of 128
            for (uint32_t i = lane; i < nv; i += 128u) {
                vec16<T> a[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) a[r] = *reinterpret_cast<const vec16<T> *>(p + (size_t)(i + 32u * r) * V);
#pragma unroll
                for (int r = 0; r < 4; ++r)
#pragma unroll
                    for (uint32_t j = 0; j < V; ++j) v += (double)prob_of(a[r].v[j]);
            }
        } else {
            for (uint32_t i = lane; i < len; i += 32u) v += (double)prob_of(p[i]);
        }
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) mass[ci] = v;
    }
}

// In place: mass[i] <- sum_{j<i} mass[j]; *total <- sum of all.  One block; thread t owns a contiguous segment.
__global__ void __launch_bounds__(1024) chunk_prefix_kernel(double *mass, uint64_t n_chunks, double *total)
{
    __shared__ double seg[1024];
    const uint64_t per = (n_chunks + 1023) / 1024, lo = min(n_chunks, (uint64_t)threadIdx.x * per), hi = min(n_chunks, lo + per);
    double s = 0.0;
    for (uint64_t i = lo; i < hi; ++i) s += mass[i];
    seg[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double run = 0.0;
        for (int t = 0; t < 1024; ++t) { const double v = seg[t]; seg[t] = run; run += v; }
        *total = run;
    }
    __syncthreads();
    double run = seg[threadIdx.x];
    for (uint64_t i = lo; i < hi; ++i) { const double v = mass[i]; mass[i] = run; run += v; }
}

template <typename T>
__global__ void __launch_bounds__(256) sample_kernel(const cx<T> *__restrict__ state, uint64_t count, uint32_t chunk_len,
                                                     const double *__restrict__ prefix, uint64_t n_chunks,
                                                     const double *__restrict__ total, const double *__restrict__ u,
                                                     uint64_t *__restrict__ out, uint32_t n_shots)
{
    const uint32_t lane = threadIdx.x & 31u, shot = blockIdx.x * 8u + (threadIdx.x >> 5);
    if (shot >= n_shots) return;
    const double target = u[shot] * *total;
    uint64_t lo = 0, hi = n_chunks;          // last chunk whose prefix is <= target
    while (hi - lo > 1) {
        const uint64_t mid = (lo + hi) >> 1;
        if (prefix[mid] <= target) lo = mid; else hi = mid;
    }
    const uint64_t base = lo * chunk_len;
    const uint32_t len = (uint32_t)min((uint64_t)chunk_len, count - base);
    double run = prefix[lo];
    uint64_t found = base + len - 1;         // rounding at the chunk end: the chunk's last amplitude
    for (uint32_t i0 = 0; i0 < len; i0 += 32u) {
        const uint32_t i = i0 + lane;
        double v = i < len ? (double)prob_of(state[base + i]) : 0.0;
        for (int o = 1; o < 32; o <<= 1) {   // inclusive scan over the 32 lanes, index order
            const double w = __shfl_up_sync(0xffffffffu, v, o);
            if ((int)lane >= o) v += w;
        }
        const unsigned hit = __ballot_sync(0xffffffffu, i < len && run + v > target);
        if (hit) { found = base + i0 + (uint32_t)(__ffs(hit) - 1); break; }
        run += __shfl_sync(0xffffffffu, v, 31);
    }
    if (lane == 0) out[shot] = found;
}

int launch_sample(int prec, const void *state, uint64_t count, double *mass, double *total, const double *u_dev,
                  uint64_t *x_dev, uint32_t n_shots, void *stream, uint64_t *launches)
{
    cudaStream_t st = (cudaStream_t)stream;
    const uint32_t chunk_len = 1u << SAMPLE_CHUNK_LOG2;
    const uint64_t n_chunks = (count + chunk_len - 1) / chunk_len;
    const uint32_t grid = (uint32_t)std::min<uint64_t>((n_chunks + 7) / 8, READOUT_BLOCKS);
    if (prec == 0) chunk_mass_kernel<float><<<grid, 256, 0, st>>>((const cx<float> *)state, count, chunk_len, mass, n_chunks);
    else chunk_mass_kernel<double><<<grid, 256, 0, st>>>((const cx<double> *)state, count, chunk_len, mass, n_chunks);
    chunk_prefix_kernel<<<1, 1024, 0, st>>>(mass, n_chunks, total);
    *launches += 2;
    if (n_shots) {
        const uint32_t g2 = (n_shots + 7) / 8;
        if (prec == 0) sample_kernel<float><<<g2, 256, 0, st>>>((const cx<float> *)state, count, chunk_len, mass, n_chunks, total, u_dev, x_dev, n_shots);
        else sample_kernel<double><<<g2, 256, 0, st>>>((const cx<double> *)state, count, chunk_len, mass, n_chunks, total, u_dev, x_dev, n_shots);
        ++*launches;
    }
    return (int)cudaGetLastError();
}

// ---- measurement-basis change for shot sampling (reading R3) ------------------------------------------
// dst = G_q src with G = H (X letter on qubit q) or H S^dagger (Y letter): (a, b) -> ((a + b') / sqrt 2, (a - b') / sqrt 2),
// b' = b for X, b' = -i b for Y.  One thread per amplitude pair; src may equal dst (each pair is owned by one thread).
template <typename T>
__global__ void __launch_bounds__(256) basis_rotate_kernel(const cx<T> *src, cx<T> *dst, uint64_t pairs, int q, int is_y)
{
    const T r = (T)0.70710678118654752440;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < pairs; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t x = ((i >> q) << (q + 1)) | (i & ((1ull << q) - 1ull));
        const cx<T> a = src[x];
        cx<T> b = src[x | (1ull << q)];
        if (is_y) b = cx<T>{b.y, -b.x};   // -i b
        dst[x] = cx<T>{(a.x + b.x) * r, (a.y + b.y) * r};
        dst[x | (1ull << q)] = cx<T>{(a.x - b.x) * r, (a.y - b.y) * r};
    }
}

int launch_basis_rotate(int prec, const void *src, void *dst, int n, int q, int is_y, void *stream, uint64_t *launches)
{
    const uint64_t pairs = 1ull << (n - 1);
    const unsigned grid = (unsigned)std::min<uint64_t>((pairs + 255) / 256, 148u * 16u);
    if (prec == 0) basis_rotate_kernel<float><<<grid, 256, 0, (cudaStream_t)stream>>>((const cx<float> *)src, (cx<float> *)dst, pairs, q, is_y);
    else basis_rotate_kernel<double><<<grid, 256, 0, (cudaStream_t)stream>>>((const cx<double> *)src, (cx<double> *)dst, pairs, q, is_y);
    ++*launches;
    return (int)cudaGetLastError();
}

// ---- diagonal energy table: scatter c at index z, then in-place Walsh-Hadamard butterflies -------
template <typename TT>
__global__ void table_scatter_kernel(TT *table, const uint64_t *__restrict__ z, const double *__restrict__ c, uint32_t count)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) table[z[i]] = (TT)c[i];
}

template <typename TT>
__global__ void __launch_bounds__(256) fwht_pass_kernel(TT *table, TileDesc td, uint32_t bitmask)
{
    extern __shared__ __align__(16) unsigned char smem[];
    TT *tile = reinterpret_cast<TT *>(smem);
    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    const int k = td.k, n_runs = td.n_runs;
    const uint64_t xbase = tile_base(blockIdx.x, td.runs, n_runs);
    for (uint32_t j = tid; j < (1u << k); j += nthr) tile[j] = table[xbase | scatter_runs(j, td.runs, n_runs)];
    __syncthreads();
    for (int p = 0; p < k; ++p) {
        if (!((bitmask >> p) & 1u)) continue;
        for (uint32_t i = tid; i < (1u << (k - 1)); i += nthr) {
            const uint32_t j = insert_zero(i, p);
            const TT u = tile[j], v = tile[j | (1u << p)];
            tile[j] = u + v;
            tile[j | (1u << p)] = u - v;
        }
        __syncthreads();
    }
    for (uint32_t j = tid; j < (1u << k); j += nthr) table[xbase | scatter_runs(j, td.runs, n_runs)] = tile[j];
}

// ================================================ launchers ===================================================
namespace {

template <typename T, int R, int MAXT>
int gate_launch_t(const GateLaunch &g, const DBlock &blk, int k, uint32_t smem_prog, int n, void *states, uint64_t stride,
                  const void *cs, int P, int batch, cudaStream_t st)
{
    DevArrays da{g.blocks, g.stages, g.ops, g.segs, g.trzs, g.tczs, g.csidx, g.ryl, g.cxs, g.slut};
    const size_t smem = HDR_BYTES + smem_prog + ((size_t)sizeof(cx<T>) << k);
    dim3 grid((unsigned)(1ull << (n - k)), (unsigned)batch);
    gate_block_kernel<T, R, MAXT><<<grid, 1u << (k - R), smem, st>>>(da, blk, (cx<T> *)states, stride, (const cx<T> *)cs, P);
    return (int)cudaGetLastError();
}

template <typename F> int set_smem(F f, int bytes)
{
    return (int)cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

}  // namespace

int kernels_init(void)
{
    const int big = 200 * 1024;
    int e = 0;
    e |= set_smem(gate_block_kernel<float, 5, 256>, big);
    e |= set_smem(gate_block_kernel<float, 5, 512>, big);
    e |= set_smem(gate_block_kernel<float, 4, 256>, big);
    e |= set_smem(gate_block_kernel<float, 4, 512>, big);
    e |= set_smem(gate_block_kernel<float, 3, 512>, big);
    e |= set_smem(gate_block_kernel<double, 4, 256>, big);
    e |= set_smem(gate_block_kernel<double, 3, 256>, big);
    e |= set_smem(gate_block_kernel<double, 3, 512>, big);
    e |= set_smem(gate_block_kernel<double, 5, 256>, big);
    e |= set_smem(expect_pass_kernel<float, float, 2>, big);
    e |= set_smem(expect_pass_kernel<float, float, 3>, big);
    e |= set_smem(expect_pass_kernel<float, float, 4>, big);
    e |= set_smem(expect_pass_kernel<float, float, 5>, big);
    e |= set_smem(expect_pass_kernel<double, double, 2>, big);
    e |= set_smem(expect_pass_kernel<double, double, 3>, big);
    e |= set_smem(expect_pass_kernel<double, double, 4>, big);
    e |= set_smem(expect_pass_kernel<double, double, 5>, big);
    e |= set_smem(fwht_pass_kernel<float>, big);
    e |= set_smem(fwht_pass_kernel<double>, big);
    return e;
}

int launch_expand_params(int prec, const double *params, void *cs, void *ry, uint64_t count, void *stream, uint64_t *launches)
{
    if (!count) return 0;
    const unsigned nb = (unsigned)((count + 255) / 256);
    cudaStream_t st = (cudaStream_t)stream;
    if (prec == 0) expand_params_kernel<float><<<nb, 256, 0, st>>>(params, (cx<float> *)cs, (ry4<float> *)ry, count);
    else expand_params_kernel<double><<<nb, 256, 0, st>>>(params, (cx<double> *)cs, (ry4<double> *)ry, count);
    ++*launches;
    return (int)cudaGetLastError();
}

int launch_init_product(int prec, const PrefixDev &pd, void *states, uint64_t stride, const void *cs, int P, int batch,
                        void *stream, uint64_t *launches)
{
    cudaStream_t st = (cudaStream_t)stream;
    dim3 grid((unsigned)(1ull << (pd.n - pd.kk)), (unsigned)batch);
    const int ntab = pd.n_vary <= 8 ? 1 : (pd.n_vary + 7) / 8;
#define GV_INIT(NT)                                                                                                       \
    do {                                                                                                                  \
        if (prec == 0) init_product_kernel<float, NT><<<grid, 256, 0, st>>>(pd, (cx<float> *)states, stride, (const cx<float> *)cs, P);      \
        else init_product_kernel<double, NT><<<grid, 256, 0, st>>>(pd, (cx<double> *)states, stride, (const cx<double> *)cs, P);             \
    } while (0)
    switch (ntab) {
    case 1: GV_INIT(1); break;
    case 2: GV_INIT(2); break;
    case 3: GV_INIT(3); break;
    case 4: GV_INIT(4); break;
    case 5: GV_INIT(5); break;
    default: return (int)cudaErrorInvalidConfiguration;
    }
#undef GV_INIT
    ++*launches;
    return (int)cudaGetLastError();
}

int launch_gate_block(int prec, int R, const GateLaunch &g, const DBlock &bi, int k, uint32_t smem_prog, int n, void *states,
                      uint64_t stride, const void *cs, int P, int batch, void *stream, uint64_t *launches)
{
    cudaStream_t st = (cudaStream_t)stream;
    const int thr = 1 << (k - R);
    ++*launches;
    if (prec == 0) {
        if (R == 5 && thr <= 256) return gate_launch_t<float, 5, 256>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
        if (R == 5 && thr <= 512) return gate_launch_t<float, 5, 512>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
        if (R == 4 && thr <= 256) return gate_launch_t<float, 4, 256>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
        if (R == 4 && thr <= 512) return gate_launch_t<float, 4, 512>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
        if (R == 3 && thr <= 512) return gate_launch_t<float, 3, 512>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
    } else {
        if (R == 4 && thr <= 256) return gate_launch_t<double, 4, 256>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
        if (R == 3 && thr <= 256) return gate_launch_t<double, 3, 256>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
        if (R == 3 && thr <= 512) return gate_launch_t<double, 3, 512>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
        if (R == 5 && thr <= 256) return gate_launch_t<double, 5, 256>(g, bi, k, smem_prog, n, states, stride, cs, P, batch, st);
    }
    --*launches;
    return (int)cudaErrorInvalidConfiguration;
}

template <typename T, typename TT>
static int expect_launch_t(const DPass *passes, int pi, int k, int n, const DGroup *groups, const DTerm *terms,
                           const void *wstat, const uint32_t *gtabs, const DRs *rss, const void *states, uint64_t stride, const void *table, double *partial, uint32_t slots_per_b,
                           uint32_t slot_off, int batch, cudaStream_t st)
{
    dim3 grid((unsigned)((1ull << (n - k)) * (uint64_t)batch));
    const size_t smem = EXPECT_HDR_BYTES + EXPECT_TAB_CAP * sizeof(cx<T>) + GT_BATCH_MAX * GT_WORDS * 4 + GT_BATCH_MAX * SGR_STRIDE + (sizeof(cx<T>) << k);
    const int TB = (k >= 11) ? 8 : (k - 3 < 5 ? 5 : k - 3);   // must match plan_expectation
    const int L = k - 1 - TB;
#define GV_EXPECT(LL)                                                                                                  \
    expect_pass_kernel<T, TT, LL><<<grid, 1 << TB, smem, st>>>(passes, pi, groups, terms, (const cx<T> *)wstat, gtabs, rss, (const cx<T> *)states, stride, \
                                                               (const TT *)table, partial, slots_per_b, slot_off, (uint32_t)batch)
    switch (L) {
    case 2: GV_EXPECT(2); break;
    case 3: GV_EXPECT(3); break;
    case 4: GV_EXPECT(4); break;
    case 5: GV_EXPECT(5); break;
    default: return (int)cudaErrorInvalidConfiguration;
    }
#undef GV_EXPECT
    return (int)cudaGetLastError();
}

int launch_expect_pass(int prec, const DPass *passes, int pi, int k, int n, const DGroup *groups, const DTerm *terms,
                       const void *wstat, const uint32_t *gtabs, const DRs *rss, const void *states, uint64_t stride, const void *table, double *partial, uint32_t slots_per_b,
                       uint32_t slot_off, int batch, void *stream, uint64_t *launches)
{
    cudaStream_t st = (cudaStream_t)stream;
    ++*launches;
    if (prec == 0)
        return expect_launch_t<float, float>(passes, pi, k, n, groups, terms, wstat, gtabs, rss, states, stride, table, partial, slots_per_b,
                                             slot_off, batch, st);
    return expect_launch_t<double, double>(passes, pi, k, n, groups, terms, wstat, gtabs, rss, states, stride, table, partial, slots_per_b,
                                           slot_off, batch, st);
}

int launch_reduce(double *partial, uint32_t slots_per_b, double *E, int batch, void *stream, uint64_t *launches)
{
    uint32_t stride = 1;
    if (slots_per_b > (1u << 16)) {   // two steps
        stride = 4096;
        dim3 grid((slots_per_b + stride - 1) / stride, (unsigned)batch);
        reduce_slices_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(partial, slots_per_b, stride);
        ++*launches;
    }
    reduce_kernel<<<batch, 256, 0, (cudaStream_t)stream>>>(partial, slots_per_b, stride, E);
    ++*launches;
    return (int)cudaGetLastError();
}

int launch_table_scatter(int prec, void *table, const uint64_t *z, const double *c, uint32_t count, void *stream,
                         uint64_t *launches)
{
    if (!count) return 0;
    const unsigned nb = (count + 255) / 256;
    if (prec == 0) table_scatter_kernel<float><<<nb, 256, 0, (cudaStream_t)stream>>>((float *)table, z, c, count);
    else table_scatter_kernel<double><<<nb, 256, 0, (cudaStream_t)stream>>>((double *)table, z, c, count);
    ++*launches;
    return (int)cudaGetLastError();
}

int launch_fwht_pass(int prec, void *table, const TileDesc &td, uint32_t bitmask, int n, void *stream, uint64_t *launches)
{
    const unsigned nb = (unsigned)(1ull << (n - td.k));
    const int thr = (1 << td.k) >= 512 ? 256 : 32;
    if (prec == 0)
        fwht_pass_kernel<float><<<nb, thr, sizeof(float) << td.k, (cudaStream_t)stream>>>((float *)table, td, bitmask);
    else
        fwht_pass_kernel<double><<<nb, thr, sizeof(double) << td.k, (cudaStream_t)stream>>>((double *)table, td, bitmask);
    ++*launches;
    return (int)cudaGetLastError();
}

}  // namespace gv
