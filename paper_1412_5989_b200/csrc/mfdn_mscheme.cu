// H1-H6: the coupled-JT -> M-scheme transformation kernels and their launchers.
//
// What one request computes:
//   3-body  v = sign * sum_J sum_{J12} sum_{J12'} cb(J12,J) ck(J12',J) * sum_{s<5} w[s] * cell[J,J12,J12'][s]
//           cb(J12,J) = <ja ma jb mb|J12 M12> <J12 M12 jc mc|J M>,  ck likewise for the ket,
//           w[s] = isospin weights of the five (T12,T12',T) combinations ("the isospin
//           coupling coefficients are precalculated with several conditionals, and the isospin loops are
//           unrolled into a single weighted summation. The core ... three nested loops over coupled
//           angular momentum values").
//   2-body  v = sign * sqrt((1+d_ab)(1+d_cd)) * sum_J cg_b(J) cg_k(J) * (w0*cell[J][0] + w1*cell[J][1])
// The slab cells of a (bra tuple, ket tuple) group are stored in exactly this loop order (A2).
#include <algorithm>
#include <cstdio>

#include "mfdn_internal.cuh"

using namespace mfdn;

namespace {

// ------------------------------------------------------------------------------- H1 decode
struct Side3 {
    int tup;       // tuple id or -1
    int ima, imb, imc;
    int tz;        // ta<<2 | tb<<1 | tc
    int twoM, twoMT, par, e;
    int sign;      // +1 / -1
    bool distinct;
};

__device__ __forceinline__ void cswap(uint32_t& ka, uint32_t& kb, uint32_t& ra, uint32_t& rb, int& sign)
{
    if (ka > kb) {
        uint32_t t = ka; ka = kb; kb = t;
        t = ra; ra = rb; rb = t;
        sign = -sign;
    }
}

// canonicalise three particles: stable sort by (orbital, SPS) ascending, sign of the permutation
__device__ __forceinline__ Side3 decode3(const Tables& T, int s0, int s1, int s2)
{
    Side3 S;
    uint32_t r0 = __ldg(T.sps_rec + s0), r1 = __ldg(T.sps_rec + s1), r2 = __ldg(T.sps_rec + s2);
    uint32_t k0 = (rec_orb(r0) << 16) | s0, k1 = (rec_orb(r1) << 16) | s1, k2 = (rec_orb(r2) << 16) | s2;
    S.distinct = (s0 != s1) && (s0 != s2) && (s1 != s2);
    S.sign = 1;
    cswap(k0, k1, r0, r1, S.sign);
    cswap(k1, k2, r1, r2, S.sign);
    cswap(k0, k1, r0, r1, S.sign);
    int a = rec_orb(r0), b = rec_orb(r1), c = rec_orb(r2);
    S.tup = __ldg(T.tuple_id3 + (a * T.n_orb + b) * T.n_orb + c);
    S.ima = rec_im(r0); S.imb = rec_im(r1); S.imc = rec_im(r2);
    S.tz = (rec_tz(r0) << 2) | (rec_tz(r1) << 1) | rec_tz(r2);
    S.twoM = 2 * (S.ima + S.imb + S.imc) - rec_twoj(r0) - rec_twoj(r1) - rec_twoj(r2);
    S.twoMT = 2 * (rec_tz(r0) + rec_tz(r1) + rec_tz(r2)) - 3;
    S.par = (rec_lpar(r0) + rec_lpar(r1) + rec_lpar(r2)) & 1;
    S.e = rec_e(r0) + rec_e(r1) + rec_e(r2);
    return S;
}

struct Side2 {
    int tup, ima, imb, tz, twoM, twoMT, par, sign;
    bool distinct;
};

__device__ __forceinline__ Side2 decode2(const Tables& T, int s0, int s1)
{
    Side2 S;
    uint32_t r0 = __ldg(T.sps_rec + s0), r1 = __ldg(T.sps_rec + s1);
    uint32_t k0 = (rec_orb(r0) << 16) | s0, k1 = (rec_orb(r1) << 16) | s1;
    S.distinct = s0 != s1;
    S.sign = 1;
    cswap(k0, k1, r0, r1, S.sign);
    S.tup = __ldg(T.tuple_id2 + rec_orb(r0) * T.n_orb + rec_orb(r1));
    S.ima = rec_im(r0); S.imb = rec_im(r1);
    S.tz = (rec_tz(r0) << 1) | rec_tz(r1);
    S.twoM = 2 * (S.ima + S.imb) - rec_twoj(r0) - rec_twoj(r1);
    S.twoMT = 2 * (rec_tz(r0) + rec_tz(r1)) - 2;
    S.par = (rec_lpar(r0) + rec_lpar(r1)) & 1;
    return S;
}

__device__ __forceinline__ bool in_range(const Tables& T, const int* s, int k)
{
    bool ok = true;
#pragma unroll
    for (int i = 0; i < 6; i++)
        if (i < k) ok = ok && ((unsigned)s[i] < (unsigned)T.n_sps);
    return ok;
}

// selection rules S1-S6 (integer only)
__device__ __forceinline__ bool select3(const Tables& T, const Side3& B, const Side3& K)
{
    return B.distinct && K.distinct && B.twoM == K.twoM && B.twoMT == K.twoMT && B.par == K.par &&
           B.e <= T.e3max && K.e <= T.e3max && B.tup >= 0 && K.tup >= 0;
}
__device__ __forceinline__ bool select2(const Side2& B, const Side2& K)
{
    return B.distinct && K.distinct && B.twoM == K.twoM && B.twoMT == K.twoMT && B.par == K.par && B.tup >= 0 &&
           K.tup >= 0;
}

// S7 helper: set of (J,T) channels in which this side has an admissible listed state
__device__ __forceinline__ unsigned long long chanmask3(const Tables& T, int4 d, int twoM12, int twoMT12)
{
    int J12min = d.y & 255, J12max = (d.y >> 8) & 255;
    unsigned long long m = 0;
    int lo = max(J12min, (abs(twoM12) + 1) >> 1);   // 2*J12 >= |2*M12|
    for (int J12 = lo; J12 <= J12max; J12++) {
        const unsigned long long* p = T.stmask3 + d.z + (J12 - J12min) * 2;
        if (twoMT12 == 0) m |= __ldg(p);
        m |= __ldg(p + 1);
    }
    return m;
}

// ------------------------------------------------------------------------------- H3-H5, 3-body
__device__ __forceinline__ double eval3(const Tables& T, const Side3& B, const Side3& K, int& mask)
{
    mask = 0;
    if (!select3(T, B, K)) return 0.0;
    const uint32_t so = __ldg(T.slab_off3 + (size_t)B.tup * T.n_tup3 + K.tup);
    if (so == NO_SLAB) return 0.0;
    const int4 db = __ldg(T.tdesc3 + B.tup), dk = __ldg(T.tdesc3 + K.tup);
    const int ja = db.x & 255, jb = (db.x >> 8) & 255, jc = (db.x >> 16) & 255;
    const int jd = dk.x & 255, je = (dk.x >> 8) & 255, jf = (dk.x >> 16) & 255;
    const int twoM12b = 2 * (B.ima + B.imb) - ja - jb, twoM12k = 2 * (K.ima + K.imb) - jd - je;
    const int tzb12 = (B.tz >> 2) + ((B.tz >> 1) & 1) - 1, tzk12 = (K.tz >> 2) + ((K.tz >> 1) & 1) - 1;  // MT12
    // S7
    const int aM = abs(B.twoM);
    unsigned long long mm = chanmask3(T, db, twoM12b, 2 * tzb12) & chanmask3(T, dk, twoM12k, 2 * tzk12);
    mm &= ~0ull << (2 * (aM >> 1));
    if (abs(B.twoMT) == 3) mm &= 0xAAAAAAAAAAAAAAAAull;
    if (mm == 0) return 0.0;
    mask = 1;
    // isospin weights
    const double* ib = T.iso3[B.tz];
    const double* ik = T.iso3[K.tz];
    const double w0 = ib[0] * ik[0], w1 = ib[0] * ik[1], w2 = ib[1] * ik[0], w3 = ib[1] * ik[1], w4 = ib[2] * ik[2];
    // stage-1 rows
    const int nj = T.nj;
    const int J12minb = db.y & 255, J12mink = dk.y & 255;
    const double* c1b = T.cg1 + __ldg(T.cg1_off + (ja >> 1) * nj + (jb >> 1)) + (B.ima * (jb + 1) + B.imb) * (min(ja, jb) + 1);
    const double* c1k = T.cg1 + __ldg(T.cg1_off + (jd >> 1) * nj + (je >> 1)) + (K.ima * (je + 1) + K.imb) * (min(jd, je) + 1);
    const double* cell = T.slab3 + (size_t)so * CELL3;
    const int Jlo = max((db.y >> 16) & 255, (dk.y >> 16) & 255), Jhi = min((db.y >> 24) & 255, (dk.y >> 24) & 255);
    double total = 0.0;
    for (int twoJ = Jlo; twoJ <= Jhi; twoJ += 2) {
        int lb = max(J12minb, abs(twoJ - jc) >> 1), hb = min((db.y >> 8) & 255, (twoJ + jc) >> 1);
        int lk = max(J12mink, abs(twoJ - jf) >> 1), hk = min((dk.y >> 8) & 255, (twoJ + jf) >> 1);
        int nb = hb - lb + 1, nk = hk - lk + 1;
        if (nb <= 0 || nk <= 0) continue;
        if (twoJ < aM) { cell += (size_t)nb * nk * CELL3; continue; }
        for (int J12 = lb; J12 <= hb; J12++) {
            double cb = 0.0;
            if (abs(twoM12b) <= 2 * J12) {
                const double* c2 = T.cg2 + __ldg(T.cg2_off + J12 * nj + (jc >> 1));
                int nJ = min(2 * J12, jc) + 1;
                cb = __ldg(c1b + (J12 - J12minb)) *
                     __ldg(c2 + (((twoM12b + 2 * J12) >> 1) * (jc + 1) + B.imc) * nJ + ((twoJ - abs(2 * J12 - jc)) >> 1));
            }
            double acc = 0.0;
            for (int J12p = lk; J12p <= hk; J12p++) {
                double ck = 0.0;
                if (abs(twoM12k) <= 2 * J12p) {
                    const double* c2 = T.cg2 + __ldg(T.cg2_off + J12p * nj + (jf >> 1));
                    int nJ = min(2 * J12p, jf) + 1;
                    ck = __ldg(c1k + (J12p - J12mink)) *
                         __ldg(c2 + (((twoM12k + 2 * J12p) >> 1) * (jf + 1) + K.imc) * nJ + ((twoJ - abs(2 * J12p - jf)) >> 1));
                }
                const double2 v01 = __ldg((const double2*)cell), v23 = __ldg((const double2*)cell + 1),
                              v45 = __ldg((const double2*)cell + 2);
                double inner = w0 * v01.x;
                inner = fma(w1, v01.y, inner);
                inner = fma(w2, v23.x, inner);
                inner = fma(w3, v23.y, inner);
                inner = fma(w4, v45.x, inner);
                acc = fma(ck, inner, acc);
                cell += CELL3;
            }
            total = fma(cb, acc, total);
        }
    }
    return (B.sign * K.sign) * total;
}

// ------------------------------------------------------------------------------- H3-H5, 2-body
__device__ __forceinline__ double eval2(const Tables& T, const Side2& B, const Side2& K, int& mask)
{
    mask = 0;
    if (!select2(B, K)) return 0.0;
    const uint32_t so = __ldg(T.slab_off2 + (size_t)B.tup * T.n_tup2 + K.tup);
    if (so == NO_SLAB) return 0.0;
    const int4 db = __ldg(T.tdesc2 + B.tup), dk = __ldg(T.tdesc2 + K.tup);
    const int aM = abs(B.twoM);
    unsigned long long mb = (unsigned long long)(uint32_t)db.z | ((unsigned long long)(uint32_t)db.w << 32);
    unsigned long long mk = (unsigned long long)(uint32_t)dk.z | ((unsigned long long)(uint32_t)dk.w << 32);
    unsigned long long mm = mb & mk & (~0ull << (2 * ((aM + 1) >> 1)));   // J >= |M|  (2J >= |2M|, 2M even)
    if (B.twoMT != 0) mm &= 0xAAAAAAAAAAAAAAAAull;                       // T = 1 only
    if (mm == 0) return 0.0;
    mask = 1;
    const int ja = db.x & 255, jb = (db.x >> 8) & 255, jc = dk.x & 255, jd = (dk.x >> 8) & 255;
    const double w0 = T.iso2[B.tz][0] * T.iso2[K.tz][0], w1 = T.iso2[B.tz][1] * T.iso2[K.tz][1];
    const int nj = T.nj;
    const int Jminb = db.y & 255, Jmink = dk.y & 255;
    const double* cb = T.cg1 + __ldg(T.cg1_off + (ja >> 1) * nj + (jb >> 1)) + (B.ima * (jb + 1) + B.imb) * (min(ja, jb) + 1);
    const double* ck = T.cg1 + __ldg(T.cg1_off + (jc >> 1) * nj + (jd >> 1)) + (K.ima * (jd + 1) + K.imb) * (min(jc, jd) + 1);
    const int Jlo = max(Jminb, Jmink), Jhi = min((db.y >> 8) & 255, (dk.y >> 8) & 255);
    const double2* cell = (const double2*)(T.slab2 + (size_t)so * CELL2);
    double total = 0.0;
    for (int J = Jlo; J <= Jhi; J++) {
        double2 v = __ldg(cell + (J - Jlo));
        double c = __ldg(cb + (J - Jminb)) * __ldg(ck + (J - Jmink));
        total = fma(c, fma(w1, v.y, w0 * v.x), total);
    }
    double norm = ((db.x >> 24) & 1) ? (((dk.x >> 24) & 1) ? 2.0 : 1.4142135623730951)
                                     : (((dk.x >> 24) & 1) ? 1.4142135623730951 : 1.0);
    return (B.sign * K.sign) * norm * total;
}

// ------------------------------------------------------------------------------- request loads
__device__ __forceinline__ void load_req3(const int32_t* req, long long r, int s[6])
{
    const int2* p = (const int2*)(req + 6 * r);
    int2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
    s[0] = a.x; s[1] = a.y; s[2] = b.x; s[3] = b.y; s[4] = c.x; s[5] = c.y;
}
__device__ __forceinline__ void load_req2(const int32_t* req, long long r, int s[6])
{
    int4 a = __ldg((const int4*)(req + 4 * r));
    s[0] = a.x; s[1] = a.y; s[2] = a.z; s[3] = a.w; s[4] = 0; s[5] = 0;
}

// ------------------------------------------------------------------------------- kernels
// Thread per request.  ORDER != nullptr: thread i handles request order[i] (after the group sort),
// so that the threads of a warp share the (bra tuple, ket tuple) slab and the loop bounds.
template <int BODY>
__global__ void __launch_bounds__(128) k_mscheme(Tables T, long long n, const int32_t* __restrict__ req,
                                                const uint32_t* __restrict__ order, double* __restrict__ out,
                                                uint8_t* __restrict__ maskout)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    long long r = order ? (long long)__ldg(order + i) : i;
    int s[6];
    if (BODY == 3) load_req3(req, r, s); else load_req2(req, r, s);
    double v = 0.0;
    int mask = 0;
    if (!in_range(T, s, 2 * BODY)) {
        atomicAdd(T.bad_count, 1ull);
    } else if (BODY == 3) {
        Side3 B = decode3(T, s[0], s[1], s[2]), K = decode3(T, s[3], s[4], s[5]);
        v = eval3(T, B, K, mask);
    } else {
        Side2 B = decode2(T, s[0], s[1]), K = decode2(T, s[2], s[3]);
        v = eval2(T, B, K, mask);
    }
    out[r] = mask ? v : 0.0;
    if (maskout) maskout[r] = (uint8_t)mask;
}

// H1 key generation (+ histogram when hist != nullptr)
template <int BODY>
__global__ void __launch_bounds__(256) k_keys(Tables T, long long n, const int32_t* __restrict__ req,
                                              uint32_t* __restrict__ keys, uint32_t* __restrict__ hist, uint32_t invalid_key,
                                              uint32_t invalid_bucket)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s[6];
    if (BODY == 3) load_req3(req, i, s); else load_req2(req, i, s);
    uint32_t key = invalid_key;
    if (in_range(T, s, 2 * BODY)) {
        if (BODY == 3) {
            Side3 B = decode3(T, s[0], s[1], s[2]), K = decode3(T, s[3], s[4], s[5]);
            if (select3(T, B, K)) key = (uint32_t)B.tup * T.n_tup3 + K.tup;
        } else {
            Side2 B = decode2(T, s[0], s[1]), K = decode2(T, s[2], s[3]);
            if (select2(B, K)) key = (uint32_t)B.tup * T.n_tup2 + K.tup;
        }
    }
    keys[i] = key;
    if (hist) atomicAdd(hist + (key == invalid_key ? invalid_bucket : key), 1u);
}

// H2: exclusive scan of the histogram (three small kernels), then scatter of request indices.
constexpr int SCAN_T = 256, SCAN_E = 16, SCAN_TILE = SCAN_T * SCAN_E;

__global__ void __launch_bounds__(SCAN_T) k_scan_tiles(uint32_t* __restrict__ data, long long m, uint32_t* __restrict__ tile_sums)
{
    __shared__ uint32_t sh[SCAN_T];
    long long base = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_E;
    uint32_t v[SCAN_E], sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_E; k++) {
        v[k] = (base + k < m) ? data[base + k] : 0u;
        sum += v[k];
    }
    sh[threadIdx.x] = sum;
    __syncthreads();
    for (int off = 1; off < SCAN_T; off <<= 1) {
        uint32_t x = threadIdx.x >= off ? sh[threadIdx.x - off] : 0u;
        __syncthreads();
        sh[threadIdx.x] += x;
        __syncthreads();
    }
    uint32_t excl = sh[threadIdx.x] - sum;
    if (threadIdx.x == SCAN_T - 1) tile_sums[blockIdx.x] = sh[threadIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_E; k++) {
        if (base + k < m) data[base + k] = excl;
        excl += v[k];
    }
}

__global__ void __launch_bounds__(1024) k_scan_sums(uint32_t* __restrict__ sums, int n_tiles)
{
    __shared__ uint32_t sh[1024];
    uint32_t carry = 0;
    for (int base = 0; base < n_tiles; base += 1024) {
        int i = base + threadIdx.x;
        uint32_t v = i < n_tiles ? sums[i] : 0u;
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int off = 1; off < 1024; off <<= 1) {
            uint32_t x = threadIdx.x >= off ? sh[threadIdx.x - off] : 0u;
            __syncthreads();
            sh[threadIdx.x] += x;
            __syncthreads();
        }
        if (i < n_tiles) sums[i] = carry + sh[threadIdx.x] - v;
        carry += sh[1023];
        __syncthreads();
    }
}

__global__ void __launch_bounds__(SCAN_T) k_scan_add(uint32_t* __restrict__ data, long long m, const uint32_t* __restrict__ tile_sums)
{
    uint32_t add = tile_sums[blockIdx.x];
    long long base = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_E;
#pragma unroll
    for (int k = 0; k < SCAN_E; k++)
        if (base + k < m) data[base + k] += add;
}

__global__ void __launch_bounds__(256) k_scatter(long long n, const uint32_t* __restrict__ keys, uint32_t* __restrict__ cursor,
                                                 uint32_t* __restrict__ order, uint32_t invalid_key, uint32_t invalid_bucket)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t key = keys[i];
    uint32_t pos = atomicAdd(cursor + (key == invalid_key ? invalid_bucket : key), 1u);
    order[pos] = (uint32_t)i;
}

size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

template <int BODY>
int run(mfdn_ctx* c, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work, size_t* work_bytes,
        uint32_t flags, void* stream)
{
    if (!c || !work_bytes || n < 0 || n >= (int64_t)0xFFFFFFF0ll) return c ? fail(c, MFDN_ERR_ARG, "bad n / work_bytes") : MFDN_ERR_ARG;
    if (BODY == 3 ? !c->has3 : !c->has2) return fail(c, MFDN_ERR_STATE, "mscheme before coupled upload");
    const long long nt = BODY == 3 ? c->t.n_tup3 : c->t.n_tup2;
    const long long n_buckets = nt * nt + 1;   // last bucket: requests failing S1-S6
    const long long n_tiles = (n_buckets + SCAN_TILE - 1) / SCAN_TILE;
    const bool sorted_path = !(flags & (MFDN_PRESORTED | MFDN_FORCE_NAIVE));
    size_t need = 256;
    size_t o_keys = 0, o_order = 0, o_hist = 0, o_sums = 0;
    if (sorted_path) {
        o_keys = 0;
        o_order = o_keys + align256((size_t)n * 4);
        o_hist = o_order + align256((size_t)n * 4);
        o_sums = o_hist + align256((size_t)n_buckets * 4);
        need = o_sums + align256((size_t)n_tiles * 4);
    }
    if (!d_work) { *work_bytes = need; return MFDN_OK; }
    if (*work_bytes < need) return fail(c, MFDN_ERR_OOM, "scratch too small");
    if (n == 0) return MFDN_OK;
    if (!d_req || !d_out) return fail(c, MFDN_ERR_ARG, "null request/output pointer");
    if (nt * nt >= 0xFFFFFFF0ll) return fail(c, MFDN_ERR_ARG, "too many tuples for 32-bit group keys");
    cudaStream_t st = (cudaStream_t)stream;
    const uint32_t* order = nullptr;
    mfdn_ctx::EvTriple ev{nullptr, nullptr, nullptr, sorted_path};
    if (c->profile) {
        cudaEvent_t* e3[3] = {&ev.a, &ev.b, &ev.c};
        for (auto pe : e3) {
            if (!c->ev_pool.empty()) { *pe = c->ev_pool.back(); c->ev_pool.pop_back(); }
            else MFDN_CUDA(c, cudaEventCreate(pe));
        }
        MFDN_CUDA(c, cudaEventRecord(ev.a, st));
    }
    if (sorted_path) {
        char* w = (char*)d_work;
        uint32_t* keys = (uint32_t*)(w + o_keys);
        uint32_t* ord = (uint32_t*)(w + o_order);
        uint32_t* hist = (uint32_t*)(w + o_hist);
        uint32_t* sums = (uint32_t*)(w + o_sums);
        MFDN_CUDA(c, cudaMemsetAsync(hist, 0, (size_t)n_buckets * 4, st));
        k_keys<BODY><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(c->t, n, d_req, keys, hist, 0xFFFFFFFFu, (uint32_t)(nt * nt));
        k_scan_tiles<<<(unsigned)n_tiles, SCAN_T, 0, st>>>(hist, n_buckets, sums);
        k_scan_sums<<<1, 1024, 0, st>>>(sums, (int)n_tiles);
        k_scan_add<<<(unsigned)n_tiles, SCAN_T, 0, st>>>(hist, n_buckets, sums);
        k_scatter<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, keys, hist, ord, 0xFFFFFFFFu, (uint32_t)(nt * nt));
        c->launches += 5;
        order = ord;
    }
    if (c->profile) MFDN_CUDA(c, cudaEventRecord(ev.b, st));
    k_mscheme<BODY><<<(unsigned)((n + 127) / 128), 128, 0, st>>>(c->t, n, d_req, order, d_out, d_mask);
    c->launches += 1;
    MFDN_CUDA(c, cudaGetLastError());
    if (c->profile) {
        MFDN_CUDA(c, cudaEventRecord(ev.c, st));
        c->ev_pending.push_back(ev);
    }
    return MFDN_OK;
}

// register-resident DFMA chains: 8 independent accumulators per thread, no memory traffic
__global__ void __launch_bounds__(256) k_fp64_peak(double* out, int iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; i++) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 12345.678) out[0] = s;   // never true; keeps the chains alive
}

}  // namespace

extern "C" int mfdn_mscheme_2b(mfdn_ctx* c, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work,
                               size_t* work_bytes, uint32_t flags, void* stream)
{
    return run<2>(c, n, d_req, d_out, d_mask, d_work, work_bytes, flags, stream);
}

extern "C" int mfdn_mscheme_3b(mfdn_ctx* c, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work,
                               size_t* work_bytes, uint32_t flags, void* stream)
{
    return run<3>(c, n, d_req, d_out, d_mask, d_work, work_bytes, flags, stream);
}

extern "C" int mfdn_group_keys(mfdn_ctx* c, int body, int64_t n, const int32_t* d_req, uint32_t* d_key, void* stream)
{
    if (!c || (body != 2 && body != 3) || n < 0 || !d_key || (n > 0 && !d_req)) return c ? fail(c, MFDN_ERR_ARG, "bad argument") : MFDN_ERR_ARG;
    if (body == 3 ? !c->has3 : !c->has2) return fail(c, MFDN_ERR_STATE, "group_keys before coupled upload");
    if (n == 0) return MFDN_OK;
    cudaStream_t st = (cudaStream_t)stream;
    if (body == 3)
        k_keys<3><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(c->t, n, d_req, d_key, nullptr, 0xFFFFFFFFu, 0u);
    else
        k_keys<2><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(c->t, n, d_req, d_key, nullptr, 0xFFFFFFFFu, 0u);
    MFDN_CUDA(c, cudaGetLastError());
    return MFDN_OK;
}

extern "C" int mfdn_profile(mfdn_ctx* c, int enable)
{
    if (!c) return MFDN_ERR_ARG;
    c->profile = enable != 0;
    return MFDN_OK;
}

extern "C" int mfdn_profile_read(mfdn_ctx* c, double* ms_sort, double* ms_transform, int64_t* calls)
{
    if (!c || !ms_sort || !ms_transform || !calls) return MFDN_ERR_ARG;
    *ms_sort = *ms_transform = 0.0;
    *calls = 0;
    for (auto& ev : c->ev_pending) {
        MFDN_CUDA(c, cudaEventSynchronize(ev.c));
        float t1 = 0.f, t2 = 0.f;
        MFDN_CUDA(c, cudaEventElapsedTime(&t1, ev.a, ev.b));
        MFDN_CUDA(c, cudaEventElapsedTime(&t2, ev.b, ev.c));
        *ms_sort += t1;
        *ms_transform += t2;
        *calls += 1;
        c->ev_pool.push_back(ev.a); c->ev_pool.push_back(ev.b); c->ev_pool.push_back(ev.c);
    }
    c->ev_pending.clear();
    return MFDN_OK;
}

extern "C" int mfdn_fp64_peak(mfdn_ctx* c, double* tflops)
{
    if (!c || !tflops) return MFDN_ERR_ARG;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    cudaEvent_t a, b;
    MFDN_CUDA(c, cudaEventCreate(&a));
    MFDN_CUDA(c, cudaEventCreate(&b));
    const int iters = 1 << 14, blocks = c->num_sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 5; rep++) {
        MFDN_CUDA(c, cudaEventRecord(a, 0));
        k_fp64_peak<<<blocks, threads>>>((double*)c->t.bad_count + 8, iters, 0.999999, 1e-9);
        MFDN_CUDA(c, cudaEventRecord(b, 0));
        MFDN_CUDA(c, cudaEventSynchronize(b));
        float ms = 0.f;
        MFDN_CUDA(c, cudaEventElapsedTime(&ms, a, b));
        double tf = 2.0 * 8.0 * iters * (double)blocks * threads / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    *tflops = best;
    return MFDN_OK;
}

// The paper's wrapper, double-buffered: chunk k uses stream k % 2.
extern "C" int mfdn_mscheme_host(mfdn_ctx* c, int body, int64_t n, const int32_t* h_req, double* h_out, uint8_t* h_mask,
                                 void* d_work, size_t* work_bytes, uint32_t flags, int64_t chunk)
{
    if (!c || !work_bytes || (body != 2 && body != 3) || n < 0 || chunk < 0) return c ? fail(c, MFDN_ERR_ARG, "bad argument") : MFDN_ERR_ARG;
    if (chunk == 0) chunk = 1 << 22;
    if (chunk > n && n > 0) chunk = n;
    const int width = 2 * body;
    size_t inner = 0;
    int rc = body == 3 ? run<3>(c, chunk, nullptr, nullptr, nullptr, nullptr, &inner, flags, nullptr)
                       : run<2>(c, chunk, nullptr, nullptr, nullptr, nullptr, &inner, flags, nullptr);
    if (rc) return rc;
    const size_t b_req = align256((size_t)chunk * width * 4), b_out = align256((size_t)chunk * 8), b_mask = align256((size_t)chunk);
    const size_t per = b_req + b_out + b_mask + align256(inner);
    if (!d_work) { *work_bytes = 2 * per; return MFDN_OK; }
    if (*work_bytes < 2 * per) return fail(c, MFDN_ERR_OOM, "scratch too small");
    if (n == 0) return MFDN_OK;
    if (!h_req || !h_out) return fail(c, MFDN_ERR_ARG, "null host pointer");
    MFDN_CUDA(c, cudaSetDevice(c->device));
    for (int k = 0; k < 2; k++)
        if (!c->hs[k]) MFDN_CUDA(c, cudaStreamCreateWithFlags(&c->hs[k], cudaStreamNonBlocking));
    int64_t k = 0;
    for (int64_t lo = 0; lo < n; lo += chunk, k++) {
        int64_t m = std::min<int64_t>(chunk, n - lo);
        cudaStream_t st = c->hs[k & 1];
        char* base = (char*)d_work + (k & 1) * per;
        int32_t* dreq = (int32_t*)base;
        double* dout = (double*)(base + b_req);
        uint8_t* dmask = (uint8_t*)(base + b_req + b_out);
        void* dw = base + b_req + b_out + b_mask;
        size_t wb = align256(inner);
        MFDN_CUDA(c, cudaMemcpyAsync(dreq, h_req + lo * width, (size_t)m * width * 4, cudaMemcpyHostToDevice, st));
        rc = body == 3 ? run<3>(c, m, dreq, dout, dmask, dw, &wb, flags, st) : run<2>(c, m, dreq, dout, dmask, dw, &wb, flags, st);
        if (rc) return rc;
        MFDN_CUDA(c, cudaMemcpyAsync(h_out + lo, dout, (size_t)m * 8, cudaMemcpyDeviceToHost, st));
        if (h_mask) MFDN_CUDA(c, cudaMemcpyAsync(h_mask + lo, dmask, (size_t)m, cudaMemcpyDeviceToHost, st));
    }
    MFDN_CUDA(c, cudaStreamSynchronize(c->hs[0]));
    MFDN_CUDA(c, cudaStreamSynchronize(c->hs[1]));
    return MFDN_OK;
}
