// Host side of libmfdn_b200.so: context, A0 orbital tables, A1 CG-table build kernel,
// A2 coupled-table upload + re-tiling kernels.  See include/mfdn_b200.h for the ABI.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>

#include "mfdn_internal.cuh"

using namespace mfdn;

namespace mfdn {
int fail(mfdn_ctx* c, int code, const std::string& msg)
{
    if (c) {
        std::lock_guard<std::mutex> lk(c->mu);
        c->err = msg;
    }
    return code;
}
int cuda_fail(mfdn_ctx* c, cudaError_t e, const char* what)
{
    if (c) {
        std::lock_guard<std::mutex> lk(c->mu);
        c->err = std::string(what) + ": " + cudaGetErrorString(e);
    }
    return e == cudaErrorMemoryAllocation ? MFDN_ERR_OOM : MFDN_ERR_CUDA;
}
}  // namespace mfdn

// One contiguous host arena -> one cudaMalloc + one cudaMemcpy (the paper's fix for its index
// array: "a single GPU allocate and GPU copy").  Offsets instead of pointers.
struct Arena {
    std::vector<char> buf;
    size_t add(const void* src, size_t bytes)
    {
        size_t off = (buf.size() + 255) & ~size_t(255);
        buf.resize(off + bytes);
        if (bytes) memcpy(buf.data() + off, src, bytes);
        return off;
    }
    template <class T>
    size_t add(const std::vector<T>& v) { return add(v.data(), v.size() * sizeof(T)); }
};

static int arena_upload(mfdn_ctx* c, Arena& a, char** dbase, cudaStream_t st)
{
    void* d = nullptr;
    MFDN_CUDA(c, cudaMalloc(&d, std::max<size_t>(a.buf.size(), 256)));
    c->owned.push_back(d);
    MFDN_CUDA(c, cudaMemcpyAsync(d, a.buf.data(), a.buf.size(), cudaMemcpyHostToDevice, st));
    MFDN_CUDA(c, cudaStreamSynchronize(st));
    *dbase = (char*)d;
    return MFDN_OK;
}

// ------------------------------------------------------------------------------------------ A0
extern "C" int mfdn_orbitals_init(mfdn_ctx** out, int device, int32_t n_orb, const int32_t* n, const int32_t* l,
                                  const int32_t* twoj, int32_t n_sps, const int32_t* sps_orb,
                                  const int32_t* sps_twom, const int32_t* sps_twotz)
{
    if (!out) return MFDN_ERR_ARG;
    *out = nullptr;
    if (!n || !l || !twoj || !sps_orb || !sps_twom || !sps_twotz) return MFDN_ERR_ARG;
    if (n_orb <= 0 || n_orb > 1023 || n_sps <= 0 || n_sps > 65535) return MFDN_ERR_ARG;
    mfdn_ctx* c = new (std::nothrow) mfdn_ctx();
    if (!c) return MFDN_ERR_OOM;
    c->device = device;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) { delete c; return MFDN_ERR_CUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) c->num_sms = prop.multiProcessorCount;
    int tjmax = 0;
    for (int o = 0; o < n_orb; o++) {
        int e_o = 2 * n[o] + l[o];
        if (n[o] < 0 || l[o] < 0 || twoj[o] < 1 || !(twoj[o] & 1) || twoj[o] > MAX_TWOJ || e_o > 63 ||
            (twoj[o] != 2 * l[o] + 1 && twoj[o] != 2 * l[o] - 1)) { delete c; return MFDN_ERR_ARG; }
        tjmax = std::max(tjmax, (int)twoj[o]);
    }
    c->orb_n.assign(n, n + n_orb);
    c->orb_l.assign(l, l + n_orb);
    c->orb_twoj.assign(twoj, twoj + n_orb);
    c->tjmax = tjmax;
    c->h_sps_rec.resize(n_sps);
    for (int s = 0; s < n_sps; s++) {
        int o = sps_orb[s];
        if (o < 0 || o >= n_orb) { delete c; return MFDN_ERR_ARG; }
        int tm = sps_twom[s], tz = sps_twotz[s];
        if (std::abs(tm) > twoj[o] || !(tm & 1) || (tz != 1 && tz != -1)) { delete c; return MFDN_ERR_ARG; }
        c->h_sps_rec[s] = sps_pack(o, (tm + twoj[o]) / 2, tz == 1, twoj[o], l[o] & 1);
    }
    void* d = nullptr;
    if (cudaMalloc(&d, n_sps * sizeof(uint32_t) + 256) != cudaSuccess) { delete c; return MFDN_ERR_OOM; }
    c->owned.push_back(d);
    if (cudaMemcpy(d, c->h_sps_rec.data(), n_sps * sizeof(uint32_t), cudaMemcpyHostToDevice) != cudaSuccess) {
        mfdn_destroy(c);
        return MFDN_ERR_CUDA;
    }
    c->t.sps_rec = (const uint32_t*)d;
    c->t.n_sps = n_sps;
    c->t.n_orb = n_orb;
    c->t.nj = (tjmax + 1) / 2;
    void* bad = nullptr;
    if (cudaMalloc(&bad, 256) != cudaSuccess) { mfdn_destroy(c); return MFDN_ERR_OOM; }
    c->owned.push_back(bad);
    cudaMemset(bad, 0, 256);
    c->t.bad_count = (unsigned long long*)bad;

    // isospin weights, "precalculated with several conditionals"; closed forms of the
    // j = 1/2 Clebsch-Gordan coefficients.
    const double r12 = std::sqrt(0.5), r13 = std::sqrt(1.0 / 3.0), r23 = std::sqrt(2.0 / 3.0);
    for (int ta = 0; ta < 2; ta++)
        for (int tb = 0; tb < 2; tb++) {
            int m12 = (ta ? 1 : -1) + (tb ? 1 : -1);  // 2*MT12
            double c0 = (m12 != 0) ? 0.0 : (ta ? r12 : -r12);  // <1/2 ta 1/2 tb|0 0>
            double c1 = (m12 != 0) ? 1.0 : r12;                // <1/2 ta 1/2 tb|1 MT12>
            c->t.iso2[ta * 2 + tb][0] = c0;
            c->t.iso2[ta * 2 + tb][1] = c1;
            for (int tc = 0; tc < 2; tc++) {
                // <1 MT12 1/2 tc|1/2 MT> and <1 MT12 1/2 tc|3/2 MT>
                double h, q;
                if (m12 == 2) { h = tc ? 0.0 : r23; q = tc ? 1.0 : r13; }
                else if (m12 == 0) { h = tc ? -r13 : r13; q = r23; }
                else { h = tc ? -r23 : 0.0; q = tc ? r13 : 1.0; }
                double* w = c->t.iso3[ta * 4 + tb * 2 + tc];
                w[0] = c0;       // (T12,T) = (0,1/2):  <0 0 1/2 tc|1/2 tc> = 1
                w[1] = c1 * h;   // (1,1/2)
                w[2] = c1 * q;   // (1,3/2)
            }
        }
    // the five 3-body weights (and two 2-body weights) per tz-bit pattern of a packed record
    std::vector<double> w3(64 * 6, 0.0), w2(16 * 2, 0.0);
    for (int tb = 0; tb < 8; tb++)
        for (int tk = 0; tk < 8; tk++) {
            const double* ib = c->t.iso3[tb];
            const double* ik = c->t.iso3[tk];
            double* w = &w3[(tb * 8 + tk) * 6];
            w[0] = ib[0] * ik[0]; w[1] = ib[0] * ik[1]; w[2] = ib[1] * ik[0]; w[3] = ib[1] * ik[1]; w[4] = ib[2] * ik[2];
        }
    for (int tb = 0; tb < 4; tb++)
        for (int tk = 0; tk < 4; tk++) {
            w2[(tb * 4 + tk) * 2 + 0] = c->t.iso2[tb][0] * c->t.iso2[tk][0];
            w2[(tb * 4 + tk) * 2 + 1] = c->t.iso2[tb][1] * c->t.iso2[tk][1];
        }
    // isospin bins: the (bra, ket) tz patterns with equal MT (1 + 9 + 9 + 1 = NBIN3), in ascending tz-bit order
    std::vector<double> wb(NBIN3 * NISO3, 0.0);
    std::vector<uint8_t> t2b(64, NBIN3 - 1);
    {
        int nbin = 0;
        for (int tb = 0; tb < 8; tb++)
            for (int tk = 0; tk < 8; tk++)
                if (__builtin_popcount(tb) == __builtin_popcount(tk)) {
                    for (int q = 0; q < NISO3; q++) wb[nbin * NISO3 + q] = w3[(tb * 8 + tk) * 6 + q];
                    t2b[tb * 8 + tk] = (uint8_t)nbin++;
                }
        if (nbin != NBIN3) { mfdn_destroy(c); return MFDN_ERR_STATE; }
    }
    void* dw = nullptr;
    const size_t nw = w3.size() + w2.size() + wb.size();
    if (cudaMalloc(&dw, nw * sizeof(double) + 64) != cudaSuccess) { mfdn_destroy(c); return MFDN_ERR_OOM; }
    c->owned.push_back(dw);
    cudaMemcpy(dw, w3.data(), w3.size() * sizeof(double), cudaMemcpyHostToDevice);
    cudaMemcpy((double*)dw + w3.size(), w2.data(), w2.size() * sizeof(double), cudaMemcpyHostToDevice);
    cudaMemcpy((double*)dw + w3.size() + w2.size(), wb.data(), wb.size() * sizeof(double), cudaMemcpyHostToDevice);
    cudaMemcpy((double*)dw + nw, t2b.data(), 64, cudaMemcpyHostToDevice);
    c->t.wtab3 = (const double*)dw;
    c->t.wtab2 = (const double*)dw + w3.size();
    c->t.wbin3 = (const double*)dw + w3.size() + w2.size();
    c->t.tz2bin3 = (const uint8_t*)((const double*)dw + nw);
    c->stage = 1;
    *out = c;
    return MFDN_OK;
}

// ------------------------------------------------------------------------------------------ A1
// Racah's closed form.  Two measures keep every entry within a few 1e-16 of the exact value
// (DESIGN.md "CG accuracy"):
//  * the alternating k-sum is rewritten over binomials,
//      sum_k (-1)^k / [k!(a-k)!(b-k)!(c-k)!(d+k)!(e+k)!]
//        = [a!(b+d)!(c+e)!]^-1 * sum_k (-1)^k C(a,k) C(b+d,b-k) C(c+e,c-k),
//    an INTEGER sum (< 2^70 for 2j <= 21) accumulated exactly in double-double, so the
//    cancellation between terms costs nothing;
//  * the prefactor sqrt(P)/[a!(b+d)!(c+e)!] is exp of a log-factorial sum carried as double-double
//    (hi+lo): the log sums reach ~150, so plain fp64 sums would lose ~3e-14.
struct dd { double hi, lo; };
__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    double s = a.hi + b.hi, bb = s - a.hi;
    double e = (a.hi - (s - bb)) + (b.hi - bb);
    double t = a.lo + b.lo, tb = t - a.lo;
    double f = (a.lo - (t - tb)) + (b.lo - tb);
    e += t;
    double s2 = s + e;
    e = e - (s2 - s);
    e += f;
    dd r;
    r.hi = s2 + e;
    r.lo = e - (r.hi - s2);
    return r;
}
__device__ __forceinline__ dd dd_neg(dd a) { return dd{-a.hi, -a.lo}; }
__device__ __forceinline__ dd dd_mul_d(dd x, double y)
{
    double p = x.hi * y;
    double e = fma(x.hi, y, -p);
    e = fma(x.lo, y, e);
    dd r;
    r.hi = p + e;
    r.lo = e - (r.hi - p);
    return r;
}

struct CgBlock { int tj1, tj2, off, count; };
constexpr int BINOM_N = 64;   // Pascal triangle rows 0..63 as doubles (exact below 2^53: rows <= 56)

__global__ void k_cg_build(const CgBlock* __restrict__ blocks, const double2* __restrict__ lfact,
                           const double* __restrict__ binom, double* __restrict__ out)
{
    CgBlock b = blocks[blockIdx.y];
    auto LF = [&](int n) { double2 v = lfact[n]; return dd{v.x, v.y}; };
    auto BIN = [&](int n, int k) { return binom[n * BINOM_N + k]; };
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < b.count; idx += gridDim.x * blockDim.x) {
        // layout [iJ][i1][i2] (projections fastest: the lanes of a warp differ only in their projections)
        int i2 = idx % (b.tj2 + 1);
        int i1 = (idx / (b.tj2 + 1)) % (b.tj1 + 1);
        int iJ = idx / ((b.tj1 + 1) * (b.tj2 + 1));
        int tJ = abs(b.tj1 - b.tj2) + 2 * iJ, tm1 = 2 * i1 - b.tj1, tm2 = 2 * i2 - b.tj2, tM = tm1 + tm2;
        double val = 0.0;
        if (abs(tM) <= tJ) {
            // all halves below are integers by construction
            int a = (b.tj1 + b.tj2 - tJ) / 2, bq = (b.tj1 - tm1) / 2, cq = (b.tj2 + tm2) / 2;
            int d = (tJ - b.tj2 + tm1) / 2, e = (tJ - b.tj1 - tm2) / 2;
            dd sum{0.0, 0.0};
            int k0 = max(0, max(-d, -e)), k1 = min(a, min(bq, cq));
            for (int k = k0; k <= k1; k++) {
                dd t{BIN(a, k), 0.0};
                t = dd_mul_d(t, BIN(bq + d, bq - k));
                t = dd_mul_d(t, BIN(cq + e, cq - k));
                sum = dd_add(sum, (k & 1) ? dd_neg(t) : t);
            }
            dd lp = LF(a);
            lp = dd_add(lp, LF((b.tj1 - b.tj2 + tJ) / 2));
            lp = dd_add(lp, LF((-b.tj1 + b.tj2 + tJ) / 2));
            lp = dd_add(lp, dd_neg(LF((b.tj1 + b.tj2 + tJ) / 2 + 1)));
            lp = dd_add(lp, LF((tJ + tM) / 2));
            lp = dd_add(lp, LF((tJ - tM) / 2));
            lp = dd_add(lp, LF(bq));
            lp = dd_add(lp, LF((b.tj1 + tm1) / 2));
            lp = dd_add(lp, LF((b.tj2 - tm2) / 2));
            lp = dd_add(lp, LF(cq));
            lp.hi *= 0.5;  // sqrt of the prefactor
            lp.lo *= 0.5;
            lp = dd_add(lp, dd_neg(LF(a)));
            lp = dd_add(lp, dd_neg(LF(bq + d)));
            lp = dd_add(lp, dd_neg(LF(cq + e)));
            val = (sum.hi + sum.lo) * (exp(lp.hi) * (1.0 + lp.lo)) * sqrt((double)(tJ + 1));
        }
        out[b.off + idx] = val;
    }
}

extern "C" int mfdn_cg_build(mfdn_ctx* c, void* stream)
{
    if (!c) return MFDN_ERR_ARG;
    if (c->stage < 1) return fail(c, MFDN_ERR_STATE, "mfdn_cg_build before mfdn_orbitals_init");
    if (c->stage >= 2) return MFDN_OK;
    cudaStream_t st = (cudaStream_t)stream;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    const int nj = c->t.nj;
    std::vector<CgBlock> blocks;
    std::vector<int32_t> off1(nj * nj), off2(2 * nj * nj);
    int64_t pos = 0;
    for (int a = 0; a < nj; a++)
        for (int b = 0; b < nj; b++) {
            int tj1 = 2 * a + 1, tj2 = 2 * b + 1;
            int cnt = (tj1 + 1) * (tj2 + 1) * (std::min(tj1, tj2) + 1);
            off1[a * nj + b] = (int32_t)pos;
            blocks.push_back({tj1, tj2, (int)pos, cnt});
            pos += cnt;
        }
    c->n_cg1 = pos;
    for (int J12 = 0; J12 < 2 * nj; J12++)
        for (int b = 0; b < nj; b++) {
            int tj1 = 2 * J12, tj2 = 2 * b + 1;
            int cnt = (tj1 + 1) * (tj2 + 1) * (std::min(tj1, tj2) + 1);
            off2[J12 * nj + b] = (int32_t)(pos - c->n_cg1);
            blocks.push_back({tj1, tj2, (int)pos, cnt});
            pos += cnt;
        }
    c->n_cg2 = pos - c->n_cg1;
    // log-factorial table as double-double, from long double accumulation of log(k)
    const int NF = 4 * (2 * nj) + 8;
    std::vector<double> lf(2 * NF);
    long double acc = 0.0L;
    for (int k = 0; k < NF; k++) {
        if (k > 1) acc += logl((long double)k);
        double hi = (double)acc;
        lf[2 * k] = hi;
        lf[2 * k + 1] = (double)(acc - (long double)hi);
    }
    std::vector<double> binom(BINOM_N * BINOM_N, 0.0);
    {
        std::vector<unsigned long long> row(BINOM_N, 0), prev(BINOM_N, 0);
        for (int nn = 0; nn < BINOM_N; nn++) {
            for (int k = 0; k <= nn; k++) row[k] = (k == 0 || k == nn) ? 1ull : prev[k - 1] + prev[k];
            for (int k = 0; k <= nn; k++) binom[nn * BINOM_N + k] = (double)row[k];
            prev.swap(row);
        }
    }
    // device layout: [stage 1 | CG_GUARD zeros | stage 2 | CG_GUARD zeros]
    void* dcg = nullptr;
    MFDN_CUDA(c, cudaMalloc(&dcg, (pos + 2 * CG_GUARD) * sizeof(double)));
    c->owned.push_back(dcg);
    MFDN_CUDA(c, cudaMemsetAsync(dcg, 0, (pos + 2 * CG_GUARD) * sizeof(double), st));
    for (size_t k = (size_t)nj * nj; k < blocks.size(); k++) blocks[k].off += CG_GUARD;
    Arena a;
    size_t o_blocks = a.add(blocks), o_lf = a.add(lf), o_off1 = a.add(off1), o_off2 = a.add(off2), o_bin = a.add(binom);
    c->h_cg2_off = off2;
    char* base = nullptr;
    int rc = arena_upload(c, a, &base, st);
    if (rc) return rc;
    dim3 grid(8, (unsigned)blocks.size());
    k_cg_build<<<grid, 128, 0, st>>>((const CgBlock*)(base + o_blocks), (const double2*)(base + o_lf),
                                     (const double*)(base + o_bin), (double*)dcg);
    MFDN_CUDA(c, cudaGetLastError());
    c->t.cg1 = (const double*)dcg;
    c->t.cg2 = (const double*)dcg + c->n_cg1 + CG_GUARD;
    c->t.cg2g = (const double*)dcg + c->n_cg1;
    c->t.cg1_off = (const int32_t*)(base + o_off1);
    c->t.cg2_off = (const int32_t*)(base + o_off2);
    c->stage = 2;
    return MFDN_OK;
}

extern "C" int mfdn_option(mfdn_ctx* c, int option, int64_t value)
{
    if (!c) return MFDN_ERR_ARG;
    if (option == MFDN_OPT_SLAB_FP32) {
        if (c->has3) return fail(c, MFDN_ERR_STATE, "MFDN_OPT_SLAB_FP32 must be set before mfdn_coupled_upload_3b");
        c->opt_slab_fp32 = value != 0;
        return MFDN_OK;
    }
    return fail(c, MFDN_ERR_ARG, "unknown option");
}

extern "C" int mfdn_cg_download(mfdn_ctx* c, int stage, double* host_out, int64_t cap, int64_t* n)
{
    if (!c || !n || (stage != 1 && stage != 2)) return MFDN_ERR_ARG;
    if (c->stage < 2) return fail(c, MFDN_ERR_STATE, "mfdn_cg_download before mfdn_cg_build");
    *n = stage == 1 ? c->n_cg1 : c->n_cg2;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    MFDN_CUDA(c, cudaDeviceSynchronize());
    if (host_out && cap >= *n)
        MFDN_CUDA(c, cudaMemcpy(host_out, stage == 1 ? c->t.cg1 : c->t.cg2, *n * sizeof(double), cudaMemcpyDeviceToHost));
    return MFDN_OK;
}

// ------------------------------------------------------------------------------------------ A2
// Re-tiling kernels: channel-major squares -> group-major slabs in kernel loop order (PAPER.md:61
// "arranged in the order that the nested loops will reference them").
struct Retile3 {
    int n_tup;
    const int4* tdesc;
    const uint4* sgrp;
    const int32_t* rowmap;
    const int32_t* chan_of;   // [(twoJ>>1)*4 + (twoT>>1)*2 + par]
    const int64_t* chan_off;
    const int32_t* chan_dim;
    const double* values;
    double* slab;
};

__device__ __forceinline__ void j12_range(int4 d, int twoJ, int& lo, int& hi)
{
    int jc = (d.x >> 16) & 255;
    lo = max(d.y & 255, abs(twoJ - jc) >> 1);
    hi = min((d.y >> 8) & 255, (twoJ + jc) >> 1);
}

__global__ void k_retile3(Retile3 p)
{
    for (long long g = blockIdx.x; g < (long long)p.n_tup * p.n_tup; g += gridDim.x) {
        uint4 sg = p.sgrp[g];
        if (sg.x == NO_SLAB) continue;
        const int gsize = (int)sg.y;
        int tb = (int)(g / p.n_tup), tk = (int)(g % p.n_tup);
        int4 db = p.tdesc[tb], dk = p.tdesc[tk];
        int par = (db.x >> 25) & 1;
        int Jlo = max((db.y >> 16) & 255, (dk.y >> 16) & 255), Jhi = min((db.y >> 24) & 255, (dk.y >> 24) & 255);
        int nJb = (((db.y >> 24) & 255) - ((db.y >> 16) & 255)) / 2 + 1, nJk = (((dk.y >> 24) & 255) - ((dk.y >> 16) & 255)) / 2 + 1;
        double* dst = p.slab + (size_t)sg.x * 2;
        for (int twoJ = Jlo; twoJ <= Jhi; twoJ += 2) {
            int lb, hb, lk, hk;
            j12_range(db, twoJ, lb, hb);
            j12_range(dk, twoJ, lk, hk);
            int nb = hb - lb + 1, nk = hk - lk + 1;
            if (nb <= 0 || nk <= 0) continue;
            int iJb = (twoJ - ((db.y >> 16) & 255)) / 2, iJk = (twoJ - ((dk.y >> 16) & 255)) / 2;
            const int pitch = row_pitch3(nk);
            for (int idx = threadIdx.x; idx < NISO3 * nb * pitch; idx += blockDim.x) {
                int slot = idx / (nb * pitch), o = idx % (nb * pitch);
                int i = o / pitch, k = o % pitch;
                double v = 0.0;
                if (k < nk) {
                    int T12 = slot >> 1 & 1, T12p = slot & 1, Ti = 0;
                    if (slot == 4) { T12 = 1; T12p = 1; Ti = 1; }
                    int ch = p.chan_of[(twoJ >> 1) * 4 + Ti * 2 + par];
                    if (ch >= 0) {
                        int r = p.rowmap[db.w + ((((lb + i) - (db.y & 255)) * 2 + T12) * nJb + iJb) * 2 + Ti];
                        int q = p.rowmap[dk.w + ((((lk + k) - (dk.y & 255)) * 2 + T12p) * nJk + iJk) * 2 + Ti];
                        if (r >= 0 && q >= 0) v = p.values[p.chan_off[ch] + (long long)r * p.chan_dim[ch] + q];
                    }
                }
                dst[(size_t)slot * gsize + o] = v;
            }
            dst += (size_t)nb * pitch;
        }
    }
}

// Isospin-combined slabs (A2; layout: vw_stride in mfdn_internal.cuh): the paper's "isospin loops ... unrolled into a
// single weighted summation" done once per (group, isospin bin, cell) at upload instead of once per
// request.  Same operation order as the kernels that sum the five planes themselves (k_transform3_small,
// k_mscheme_naive use w0*p0, then fma over s = 1..4), so a value does not depend on the path its group takes.
__global__ void k_vw20(long long n_groups, const uint4* __restrict__ sgrp, const double* __restrict__ slab,
                       const double* __restrict__ wbin, uint32_t* __restrict__ vw20, int f32)
{
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const uint4 sg = sgrp[g];
        if (sg.x == NO_SLAB) continue;
        const uint32_t gsize = sg.y, S = vw_stride(gsize, f32);
        const double* src = slab + (size_t)sg.x * 2;
        uint32_t* dst = vw20 + (size_t)sg.z * 4;
        for (uint32_t idx = threadIdx.x; idx < NBIN3 * gsize; idx += blockDim.x) {
            const uint32_t b = idx / gsize, cell = idx - b * gsize;
            const double* w = wbin + b * NISO3;
            double v = w[0] * src[cell];
            v = fma(w[1], src[gsize + cell], v);
            v = fma(w[2], src[2 * (size_t)gsize + cell], v);
            v = fma(w[3], src[3 * (size_t)gsize + cell], v);
            v = fma(w[4], src[4 * (size_t)gsize + cell], v);
            if (f32) {   // footprint variant: the combined value rounded to fp32 (arithmetic stays fp64)
                dst[(size_t)b * S + cell] = __float_as_uint((float)v);
            } else {
                dst[(size_t)b * S + cell] = (uint32_t)__double2loint(v);
                dst[(size_t)b * S + gsize + cell] = (uint32_t)__double2hiint(v);
            }
        }
        for (uint32_t b = threadIdx.x; b < NBIN3; b += blockDim.x)
            if (!f32 || !(gsize & 1u)) dst[(size_t)b * S + (f32 ? gsize : 2 * gsize)] = 0u;   // the pad word, if there is one
    }
}

// Per-tuple coefficient tables (A1/A2), one block per J of the tuple: dtab[tk.x + block(J) + sigma(ima, imb, imc)*nb(J) + i] =
// <ja ma jb mb|J12 M12> <J12 M12 jc mc|J M> for the tuple's rows (J, J12) in loop order; one fp64 product of the two
// tabulated coefficients, 0 where |M12| > J12 or |M| > J (the zero guard of the stage-2 table).
struct Dtab3 {
    const int4* tdesc;
    const int4* tk;
    const int2* trow;      // {first row of the tuple in rowtab, -}
    const int2* rowtab;    // per row {cg2g offset at A = 0, cg1 offset relative to the m-pair base}
    const int2* rowdst;    // per row {offset of its J block in the tuple's table, rows of the block << 8 | row within the block}
    const int32_t* nrows;
    const uint16_t* sig;
    const int32_t* sigoff;
    const double* cg1;
    const int32_t* cg1_off;
    const double* cg2g;
    int nj;
    double* dtab;
};

__global__ void k_dtab3(Dtab3 p)
{
    const int t = blockIdx.x;
    const int4 d = p.tdesc[t], k = p.tk[t];
    const int ja = d.x & 255, jb = (d.x >> 8) & 255, jc = (d.x >> 16) & 255;
    const int S = k.y, nr = p.nrows[t], r0 = p.trow[t].x;
    const int c1 = p.cg1_off[(ja >> 1) * p.nj + (jb >> 1)];
    for (int idx = threadIdx.x; idx < nr * S; idx += blockDim.x) {
        int r = idx / S, o = idx % S;
        int imc = o % (jc + 1), imb = (o / (jc + 1)) % (jb + 1), ima = o / ((jc + 1) * (jb + 1));
        int2 rt = p.rowtab[r0 + r];
        int A = (ima + imb - ((ja + jb) >> 1)) * (jc + 1) + imc;
        int2 rd = p.rowdst[r0 + r];
        p.dtab[(size_t)(uint32_t)k.x + (size_t)rd.x + (size_t)p.sig[p.sigoff[t] + o] * (rd.y >> 8) + (rd.y & 255)] =
            p.cg1[c1 + ima * (jb + 1) + imb + rt.y] * p.cg2g[rt.x + A];
    }
}

struct Retile2 {
    int n_tup;
    const int4* tdesc;
    const uint32_t* slab_off;
    const int32_t* rowmap;
    const int32_t* rowmap_off;
    const int32_t* chan_of;   // [J*4 + T*2 + par]
    const int64_t* chan_off;
    const int32_t* chan_dim;
    const double* values;
    double* slab;
};

__global__ void k_retile2(Retile2 p)
{
    long long total = (long long)p.n_tup * p.n_tup;
    for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < total; g += (long long)gridDim.x * blockDim.x) {
        uint32_t so = p.slab_off[g];
        if (so == NO_SLAB) continue;
        int tb = (int)(g / p.n_tup), tk = (int)(g % p.n_tup);
        int4 db = p.tdesc[tb], dk = p.tdesc[tk];
        int par = (db.x >> 25) & 1;
        int Jlo = max(db.y & 255, dk.y & 255), Jhi = min((db.y >> 8) & 255, (dk.y >> 8) & 255);
        double* dst = p.slab + (size_t)so * CELL2;
        for (int J = Jlo; J <= Jhi; J++)
            for (int T = 0; T < 2; T++) {
                double v = 0.0;
                int ch = p.chan_of[J * 4 + T * 2 + par];
                if (ch >= 0) {
                    int r = p.rowmap[p.rowmap_off[tb] + (J - (db.y & 255)) * 2 + T];
                    int q = p.rowmap[p.rowmap_off[tk] + (J - (dk.y & 255)) * 2 + T];
                    if (r >= 0 && q >= 0) v = p.values[p.chan_off[ch] + (long long)r * p.chan_dim[ch] + q];
                }
                *dst++ = v;
            }
    }
}

static int stage_values(mfdn_ctx* c, const double* values, int on_device, int64_t count, cudaStream_t st,
                        const double** dvals, void** tmp)
{
    *tmp = nullptr;
    if (on_device) { *dvals = values; return MFDN_OK; }
    MFDN_CUDA(c, cudaMalloc(tmp, std::max<int64_t>(count, 1) * sizeof(double)));
    MFDN_CUDA(c, cudaMemcpyAsync(*tmp, values, count * sizeof(double), cudaMemcpyHostToDevice, st));
    *dvals = (const double*)*tmp;
    return MFDN_OK;
}

extern "C" int mfdn_coupled_upload_3b(mfdn_ctx* c, int32_t e3max, int32_t n_chan, const int32_t* chan_twoJ,
                                      const int32_t* chan_twoT, const int32_t* chan_par, const int32_t* chan_dim,
                                      const int64_t* chan_off, const int32_t* state_a, const int32_t* state_b,
                                      const int32_t* state_c, const int32_t* state_J12, const int32_t* state_T12,
                                      const double* values, int values_on_device, void* stream)
{
    if (!c) return MFDN_ERR_ARG;
    if (c->stage < 2) return fail(c, MFDN_ERR_STATE, "mfdn_coupled_upload_3b before mfdn_cg_build");
    if (c->has3) return fail(c, MFDN_ERR_STATE, "3-body table already uploaded");
    if (n_chan <= 0 || !chan_twoJ || !chan_twoT || !chan_par || !chan_dim || !chan_off || !state_a || !state_b ||
        !state_c || !state_J12 || !state_T12 || !values || e3max < 0)
        return fail(c, MFDN_ERR_ARG, "null or empty argument");
    cudaStream_t st = (cudaStream_t)stream;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    const int No = c->t.n_orb;
    const auto& tj = c->orb_twoj;
    // ---- validate channels, collect tuples
    std::vector<int32_t> chan_of(32 * 4, -1);
    int64_t n_states = 0, n_values = 0;
    for (int ch = 0; ch < n_chan; ch++) {
        int J = chan_twoJ[ch], T = chan_twoT[ch], P = chan_par[ch];
        if (J < 1 || !(J & 1) || J > 3 * MAX_TWOJ || (T != 1 && T != 3) || (P != 0 && P != 1) || chan_dim[ch] < 0 || chan_off[ch] < 0)
            return fail(c, MFDN_ERR_TABLE, "bad channel quantum numbers");
        int32_t& slot = chan_of[(J >> 1) * 4 + (T >> 1) * 2 + P];
        if (slot >= 0) return fail(c, MFDN_ERR_TABLE, "duplicate channel");
        slot = ch;
        n_states += chan_dim[ch];
        n_values = std::max<int64_t>(n_values, chan_off[ch] + (int64_t)chan_dim[ch] * chan_dim[ch]);
    }
    std::vector<int64_t> tkeys;
    tkeys.reserve(n_states);
    {
        int64_t s = 0;
        for (int ch = 0; ch < n_chan; ch++)
            for (int r = 0; r < chan_dim[ch]; r++, s++) {
                int a = state_a[s], b = state_b[s], cc = state_c[s], J12 = state_J12[s], T12 = state_T12[s];
                if (a < 0 || a > b || b > cc || cc >= No) return fail(c, MFDN_ERR_TABLE, "state orbitals not a<=b<=c in range");
                int e = 2 * (c->orb_n[a] + c->orb_n[b] + c->orb_n[cc]) + c->orb_l[a] + c->orb_l[b] + c->orb_l[cc];
                if (e > e3max) return fail(c, MFDN_ERR_TABLE, "state above E3max");
                if (((c->orb_l[a] + c->orb_l[b] + c->orb_l[cc]) & 1) != chan_par[ch]) return fail(c, MFDN_ERR_TABLE, "state parity != channel parity");
                if (T12 < 0 || T12 > 1 || 2 * J12 < std::abs(tj[a] - tj[b]) || 2 * J12 > tj[a] + tj[b])
                    return fail(c, MFDN_ERR_TABLE, "J12/T12 triangle");
                if (a == b && !((J12 + T12) & 1)) return fail(c, MFDN_ERR_TABLE, "a==b needs J12+T12 odd");
                if (chan_twoJ[ch] < std::abs(2 * J12 - tj[cc]) || chan_twoJ[ch] > 2 * J12 + tj[cc]) return fail(c, MFDN_ERR_TABLE, "J triangle");
                if (chan_twoT[ch] < std::abs(2 * T12 - 1) || chan_twoT[ch] > 2 * T12 + 1) return fail(c, MFDN_ERR_TABLE, "T triangle");
                tkeys.push_back(((int64_t)a * No + b) * No + cc);
            }
    }
    std::vector<int64_t> tuples = tkeys;
    std::sort(tuples.begin(), tuples.end());
    tuples.erase(std::unique(tuples.begin(), tuples.end()), tuples.end());
    const int nt = (int)tuples.size();
    if (nt == 0) return fail(c, MFDN_ERR_TABLE, "empty table");
    std::vector<int32_t> tuple_id((size_t)No * No * No, -1);
    std::vector<int4> tdesc(nt);
    std::vector<int32_t> nJ12v(nt), nJv(nt);
    size_t rm_size = 0, sm_size = 0;
    for (int t = 0; t < nt; t++) {
        int64_t k = tuples[t];
        int a = (int)(k / ((int64_t)No * No)), b = (int)((k / No) % No), cc = (int)(k % No);
        tuple_id[k] = t;
        int ja = tj[a], jb = tj[b], jc = tj[cc];
        int J12min = std::abs(ja - jb) / 2, J12max = (ja + jb) / 2;
        int twoJmin = 1 << 30;
        for (int J12 = J12min; J12 <= J12max; J12++) twoJmin = std::min(twoJmin, std::abs(2 * J12 - jc));
        int twoJmax = ja + jb + jc;
        int par = (c->orb_l[a] + c->orb_l[b] + c->orb_l[cc]) & 1;
        nJ12v[t] = J12max - J12min + 1;
        nJv[t] = (twoJmax - twoJmin) / 2 + 1;
        tdesc[t].x = ja | (jb << 8) | (jc << 16) | ((a == b) << 24) | (par << 25);
        tdesc[t].y = J12min | (J12max << 8) | (twoJmin << 16) | (twoJmax << 24);
        tdesc[t].z = (int)sm_size;
        tdesc[t].w = (int)rm_size;
        sm_size += (size_t)nJ12v[t] * 2;
        rm_size += (size_t)nJ12v[t] * 2 * nJv[t] * 2;
    }
    std::vector<int32_t> rowmap(rm_size, -1);
    std::vector<unsigned long long> stmask(sm_size, 0ull);
    {
        int64_t s = 0;
        for (int ch = 0; ch < n_chan; ch++)
            for (int r = 0; r < chan_dim[ch]; r++, s++) {
                int t = tuple_id[tkeys[s]];
                int4 d = tdesc[t];
                int i12 = state_J12[s] - (d.y & 255), T12 = state_T12[s];
                int iJ = (chan_twoJ[ch] - ((d.y >> 16) & 255)) / 2, Ti = chan_twoT[ch] >> 1;
                int32_t& slot = rowmap[d.w + ((size_t)(i12 * 2 + T12) * nJv[t] + iJ) * 2 + Ti];
                if (slot >= 0) return fail(c, MFDN_ERR_TABLE, "duplicate state in channel");
                slot = r;
                stmask[d.z + i12 * 2 + T12] |= 1ull << ((chan_twoJ[ch] >> 1) * 2 + Ti);
            }
    }
    // stmask -> suffix OR over J12 (per T12): entry [i12][T12] = channels of all listed states with J12 >= J12min + i12,
    // so that S7's "some admissible J12 >= |M12|" is ONE 16-byte look-up per side
    for (int t = 0; t < nt; t++)
        for (int i = nJ12v[t] - 2; i >= 0; i--)
            for (int T12 = 0; T12 < 2; T12++) stmask[tdesc[t].z + i * 2 + T12] |= stmask[tdesc[t].z + (i + 1) * 2 + T12];
    // tuples with identical mask rows share one copy (a complete table has one per (ja, jb, jc, a == b) class): k_keys3s keeps
    // the deduplicated array in shared memory
    {
        std::map<std::vector<unsigned long long>, int> seen;
        std::vector<unsigned long long> packed;
        for (int t = 0; t < nt; t++) {
            std::vector<unsigned long long> rows(stmask.begin() + tdesc[t].z, stmask.begin() + tdesc[t].z + (size_t)nJ12v[t] * 2);
            auto it = seen.find(rows);
            if (it == seen.end()) {
                it = seen.emplace(rows, (int)packed.size()).first;
                packed.insert(packed.end(), rows.begin(), rows.end());
            }
            tdesc[t].z = it->second;
        }
        stmask.swap(packed);
    }
    // The same look-up with the arithmetic done here: per tuple, indexed by [ima + imb][MT12 == 0], the channel set of all listed
    // states with J12 >= |M12| and an admissible T12 (T12 = 0 only if MT12 = 0).  k_keys3s keeps this table in shared memory: S7 is
    // then one 8-byte look-up per side without the J12-range arithmetic (22 -> 6 instructions per side).  Shared by content.
    std::vector<unsigned long long> stm12;
    std::vector<int32_t> stm12_off(nt);
    {
        std::map<std::array<int, 4>, int> seen;
        for (int t = 0; t < nt; t++) {
            const int4 d = tdesc[t];
            const int jab = (d.x & 255) + ((d.x >> 8) & 255), J12min = d.y & 255, J12max = (d.y >> 8) & 255;
            const std::array<int, 4> key{d.z, jab, J12min, J12max};
            auto it = seen.find(key);
            if (it == seen.end()) {
                it = seen.emplace(key, (int)stm12.size()).first;
                for (int i12 = 0; i12 <= jab; i12++) {
                    const int lo = std::max(J12min, (std::abs(2 * i12 - jab) + 1) >> 1);
                    for (int e = 0; e < 2; e++) {
                        unsigned long long m = 0ull;
                        if (lo <= J12max) m = (e ? stmask[d.z + (size_t)(lo - J12min) * 2] : 0ull) | stmask[d.z + (size_t)(lo - J12min) * 2 + 1];
                        stm12.push_back(m);
                    }
                }
            }
            stm12_off[t] = it->second;
        }
    }
    auto range = [&](int4 d, int twoJ, int& lo, int& hi) {
        int jc = (d.x >> 16) & 255;
        lo = std::max(d.y & 255, std::abs(twoJ - jc) >> 1);
        hi = std::min((d.y >> 8) & 255, (twoJ + jc) >> 1);
    };
    // ---- row tables (A2 "tile index": flat offsets, no pointers -- PAPER.md:109-121).  Per (tuple, J, J12) row the
    //      request-independent parts of the two coefficient addresses (used only to build dtab3):
    //        x: <J12 M12 jc mc|J M> lives at cg2g[x + A],  A = M12*(jc+1) + imc  (x includes CG_GUARD and J12*(jc+1))
    //        y: <ja ma jb mb|J12 M12> lives at cg1[c1 + y],  c1 = off(ja,jb) + ima*(jb+1) + imb
    //      and per (tuple, J): {offset of the J block in the tuple's coefficient table, number of rows nb(J)}.  Inside a
    //      block the nb coefficients of one m-state are contiguous ([sigma][row]): a request reads all its coefficients of
    //      a J block with one address computation and vector loads, and neighbouring m-states stay neighbours in memory.
    std::vector<int2> trow(nt), rowtab, rowdst, jinfo;
    std::vector<int4> tk(nt);
    std::vector<int32_t> nrows(nt), sigoff(nt), mstoff(nt);
    std::vector<uint16_t> sig, isig, mstart;   // mstart: per tuple, first sigma of every iM (prefix counts; sumj + 2 entries)
    uint64_t dtab_len = 0;
    // Everything built in this loop -- rows, J blocks, sigma order, the coefficient table -- depends on the tuple only through
    // (ja, jb, jc) (the J12 and J ranges above are the triangle ranges, not the listed states): tuples of one j-class share
    // one copy (config 3: 590 tuples, 84 classes; the coefficient tables shrink from 4.1 MB to 0.6 MB and the sigma maps fit
    // in shared memory).  nrows = 0 marks the tuples that are not the first of their class for k_dtab3.
    std::vector<int32_t> class_rep(1 << 15, -1);   // (ja, jb, jc), 2j <= 21 < 32 each
    for (int t = 0; t < nt; t++) {
        int4 d = tdesc[t];
        int ja = d.x & 255, jb = (d.x >> 8) & 255, jc = (d.x >> 16) & 255;
        int32_t& first = class_rep[ja | (jb << 5) | (jc << 10)];
        if (first >= 0) {
            trow[t] = trow[first];
            nrows[t] = 0;
            sigoff[t] = sigoff[first];
            mstoff[t] = mstoff[first];
            tk[t] = tk[first];
            continue;
        }
        first = t;
        trow[t].x = (int)rowtab.size();
        trow[t].y = (int)jinfo.size();
        const int S = (ja + 1) * (jb + 1) * (jc + 1);
        if (S > MAX_STATES3) return fail(c, MFDN_ERR_TABLE, "tuple with more than 4096 m-states");
        uint64_t tlen = 0;   // doubles of this tuple's table so far (every block starts 16-byte aligned)
        for (int twoJ = (d.y >> 16) & 255; twoJ <= ((d.y >> 24) & 255); twoJ += 2) {
            int lo, hi;
            range(d, twoJ, lo, hi);
            int2 ji;
            ji.x = (int)tlen;
            ji.y = std::max(0, hi - lo + 1);
            if (ji.y > 255) return fail(c, MFDN_ERR_TABLE, "more than 255 J12 values in one J block");
            jinfo.push_back(ji);
            for (int J12 = lo; J12 <= hi; J12++) {
                int iJ = (twoJ - std::abs(2 * J12 - jc)) / 2;
                int2 e;
                e.x = CG_GUARD + c->h_cg2_off[J12 * c->t.nj + (jc >> 1)] + (iJ * (2 * J12 + 1) + J12) * (jc + 1);
                e.y = (J12 - (d.y & 255)) * (ja + 1) * (jb + 1);
                rowtab.push_back(e);
                rowdst.push_back(int2{ji.x, (ji.y << 8) | (J12 - lo)});
            }
            tlen = (tlen + (uint64_t)S * ji.y + 1) & ~1ull;
        }
        nrows[t] = (int)rowtab.size() - trow[t].x;
        // sigma: m-states of the tuple ordered by (iM = ima+imb+imc, ima, imb); counting sort over iM
        sigoff[t] = (int32_t)sig.size();
        {
            std::vector<int> start(ja + jb + jc + 2, 0);
            for (int a = 0; a <= ja; a++) for (int b = 0; b <= jb; b++) for (int m = 0; m <= jc; m++) start[a + b + m + 1]++;
            for (size_t i = 1; i < start.size(); i++) start[i] += start[i - 1];
            mstoff[t] = (int32_t)mstart.size();
            for (int v : start) mstart.push_back((uint16_t)v);
            sig.resize(sig.size() + S);
            isig.resize(sig.size());
            uint16_t* sg = sig.data() + sigoff[t];
            uint16_t* isg = isig.data() + sigoff[t];   // sigma -> natural index (block mode needs the m's of a row)
            for (int a = 0; a <= ja; a++) for (int b = 0; b <= jb; b++) for (int m = 0; m <= jc; m++) {
                const int nat = (a * (jb + 1) + b) * (jc + 1) + m;
                sg[nat] = (uint16_t)start[a + b + m]++;
                isg[sg[nat]] = (uint16_t)nat;
            }
        }
        if (dtab_len + tlen >= 0x7FFFFFF0ull) return fail(c, MFDN_ERR_OOM, "coefficient table too large for 31-bit offsets");
        tk[t].x = (int)dtab_len;
        tk[t].y = S;
        tk[t].z = trow[t].y;
        tk[t].w = (ja + jb + jc) | (d.y & 0xFFFF0000);
        dtab_len += tlen;
    }
    // ---- group descriptors: slab offset (16-byte units) and plane size, rows in loop order J, J12
    //      and the (group, M) buckets of the request sort: every same-parity group owns one bucket per common M
    const int f32 = c->opt_slab_fp32 ? 1 : 0;
    std::vector<uint4> sgrp((size_t)nt * nt, uint4{NO_SLAB, 0u, 0u, 0u});
    std::vector<uint32_t> gbase((size_t)nt * nt + 1, 0u);
    uint64_t cells = 0;   // in 16-byte units
    uint64_t vwcells = 0; // 16-byte units of the isospin-combined slabs
    uint64_t buckets = 0;
    for (int tb = 0; tb < nt; tb++)
        for (int tkk = 0; tkk < nt; tkk++) {
            int4 db = tdesc[tb], dk = tdesc[tkk];
            gbase[(size_t)tb * nt + tkk] = (uint32_t)buckets;
            if (((db.x ^ dk.x) >> 25) & 1) continue;
            {
                const int sb = (db.x & 255) + ((db.x >> 8) & 255) + ((db.x >> 16) & 255);
                const int sk = (dk.x & 255) + ((dk.x >> 8) & 255) + ((dk.x >> 16) & 255);
                buckets += (uint64_t)std::min(sb, sk) + 1;
                if (buckets >= (uint64_t)REC_INVALID) return fail(c, MFDN_ERR_OOM, "too many (group, M) buckets for 27-bit sort keys");
            }
            int Jlo = std::max((db.y >> 16) & 255, (dk.y >> 16) & 255), Jhi = std::min((db.y >> 24) & 255, (dk.y >> 24) & 255);
            uint64_t gsize = 0;
            for (int twoJ = Jlo; twoJ <= Jhi; twoJ += 2) {
                int lb, hb, lk, hk;
                range(db, twoJ, lb, hb);
                range(dk, twoJ, lk, hk);
                if (hb >= lb && hk >= lk) gsize += (uint64_t)(hb - lb + 1) * row_pitch3(hk - lk + 1);
            }
            if (gsize == 0) continue;
            const uint64_t vw16 = ((uint64_t)NBIN3 * vw_stride((uint32_t)gsize, f32) + 3) / 4;   // 16-byte units, rounded up
            if (cells + gsize * NISO3 / 2 >= 0xFFFFFFF0ull || vwcells + vw16 >= 0xFFFFFFF0ull)
                return fail(c, MFDN_ERR_OOM, "table too large for 32-bit slab offsets");
            // dense-block path (H5'): feasible if every (M) block of m-states fits one warp's tile buffer and the
            // flattened ket rows fit its row map; w = feasible << 31 | number of (bra, ket) m-state pairs with equal M
            uint32_t dense = 0u;
            {
                const int sb = (db.x & 255) + ((db.x >> 8) & 255) + ((db.x >> 16) & 255);
                const int sk = (dk.x & 255) + ((dk.x >> 8) & 255) + ((dk.x >> 16) & 255);
                const int mm = std::min(sb, sk);
                const uint16_t* msb = mstart.data() + mstoff[tb];
                const uint16_t* msk = mstart.data() + mstoff[tkk];
                uint64_t pairs = 0;
                bool ok = true;
                for (int mi = 0; mi <= mm; mi++) {
                    const int ib = mi + (sb - mm) / 2, ik = mi + (sk - mm) / 2;
                    const int nmb = msb[ib + 1] - msb[ib], nmk = msk[ik + 1] - msk[ik];
                    pairs += (uint64_t)nmb * nmk;
                    if (((nmb + 7) & ~7) * ((nmk + 7) & ~7) > DENSE_CAP) ok = false;
                }
                int rk = 0;
                for (int twoJ = Jlo; twoJ <= Jhi; twoJ += 2) {
                    int lk, hk;
                    range(dk, twoJ, lk, hk);
                    rk += std::max(0, hk - lk + 1);
                }
                if (rk > DENSE_RMAX) ok = false;
                dense = (ok ? 0x80000000u : 0u) | (uint32_t)std::min<uint64_t>(pairs, 0x7FFFFFFFull);
            }
            sgrp[(size_t)tb * nt + tkk] = uint4{(uint32_t)cells, (uint32_t)gsize, (uint32_t)vwcells, dense};
            cells += gsize * NISO3 / 2;
            vwcells += vw16;
        }
    gbase[(size_t)nt * nt] = (uint32_t)buckets;
    // The same bucket numbers from two small tables (k_keys keeps them in shared memory instead of gathering from the
    // n_tup^2 array): gbase[b][k] = rowbase[b] + colcum[class(b)][k], class = (ja+jb+jc, parity) of the bra tuple, because
    // the buckets a ket adds to a bra's row depend on the bra only through that pair.  class id in bits 26..30 of tdesc.x.
    std::vector<uint32_t> rowbase(nt, 0u);
    std::vector<uint16_t> colcum;
    int ncls = 0;
    {
        std::vector<int> cls_of(128, -1);   // (sumj, par) -> class
        std::vector<uint32_t> rowtotal;
        bool fits = true;
        for (int t = 0; t < nt; t++) {
            const int sj = (tdesc[t].x & 255) + ((tdesc[t].x >> 8) & 255) + ((tdesc[t].x >> 16) & 255), par = (tdesc[t].x >> 25) & 1;
            int& cl = cls_of[sj * 2 + par];
            if (cl < 0) {
                cl = ncls++;
                colcum.resize((size_t)ncls * nt);
                uint32_t run = 0;
                for (int k = 0; k < nt; k++) {
                    if (run > 65535u) fits = false;
                    colcum[(size_t)cl * nt + k] = (uint16_t)run;
                    const int sk = (tdesc[k].x & 255) + ((tdesc[k].x >> 8) & 255) + ((tdesc[k].x >> 16) & 255);
                    if (((tdesc[k].x >> 25) & 1) == par) run += (uint32_t)std::min(sj, sk) + 1u;
                }
                rowtotal.push_back(run);
            }
            tdesc[t].x |= cl << 26;
        }
        uint64_t run = 0;
        for (int t = 0; t < nt; t++) {
            rowbase[t] = (uint32_t)run;
            run += rowtotal[(tdesc[t].x >> 26) & 31];
        }
        if (!fits || ncls > 31) { ncls = 0; colcum.assign(1, 0); }   // k_keys then reads gbase3
    }
    // ---- one arena for the resident index tables, one for the upload-only ones
    Arena res, tmp;
    // (a,b) -> tuple map: the sorted tuple list keeps the tuples of one (a,b) together with ascending c; if every such run
    // is a dense c range (true for any E3max truncation of an energy-ordered orbital list) k_keys finds a tuple with one
    // 8-byte shared-memory look-up instead of a random read of the n_orb^3 table
    std::vector<int2> ab((size_t)No * No, int2{-1, 0});
    bool ab_dense = No * No <= 65535 * 16;
    for (int t = 0; t < nt && ab_dense; t++) {
        int64_t k = tuples[t];
        int a = (int)(k / ((int64_t)No * No)), b = (int)((k / No) % No), cc = (int)(k % No);
        int2& e = ab[(size_t)a * No + b];
        if (e.x < 0) { e.x = t; e.y = cc | (1 << 16); }
        else if (cc == (e.y & 0xFFFF) + (e.y >> 16) && (e.y >> 16) < 32767) e.y += 1 << 16;
        else ab_dense = false;
    }
    std::vector<int4> tdesc_rt = tdesc;   // run-time copy: w = start of the tuple's sigma table (the row-map offset is upload-only)
    for (int t = 0; t < nt; t++) tdesc_rt[t].w = sigoff[t];
    size_t o_tid = res.add(tuple_id), o_desc_rt = res.add(tdesc_rt), o_sgrp = res.add(sgrp), o_sm = res.add(stmask);
    size_t o_sm12 = res.add(stm12), o_sm12off = res.add(stm12_off);
    size_t o_gbase = res.add(gbase), o_rowbase = res.add(rowbase), o_colcum = res.add(colcum);
    size_t o_desc = tmp.add(tdesc), o_ab = res.add(ab);
    size_t o_tk = res.add(tk), o_jinfo = res.add(jinfo), o_sig = res.add(sig), o_sigoff = res.add(sigoff);
    size_t o_mstart = res.add(mstart), o_mstoff = res.add(mstoff);
    // block mode (NEXT-2): sigma -> m's, tuple -> orbitals, (orbital, tz, m index) -> SPS index or -1
    std::vector<int4> torb(nt);
    for (int t = 0; t < nt; t++) {
        const int64_t k = tuples[t];
        torb[t] = int4{(int)(k / ((int64_t)No * No)), (int)((k / No) % No), (int)(k % No), 0};
    }
    std::vector<int32_t> spsidx((size_t)No * 64, -1);
    for (int sp = 0; sp < c->t.n_sps; sp++) {
        const uint32_t r = c->h_sps_rec[sp];
        spsidx[((size_t)rec_orb(r) * 2 + rec_tz(r)) * 32 + rec_im(r)] = sp;
    }
    size_t o_isig = res.add(isig), o_torb = res.add(torb), o_spsidx = res.add(spsidx);
    std::vector<int64_t> coff(chan_off, chan_off + n_chan);
    std::vector<int32_t> cdim(chan_dim, chan_dim + n_chan);
    size_t o_rm = tmp.add(rowmap), o_cof = tmp.add(chan_of), o_coff = tmp.add(coff), o_cdim = tmp.add(cdim);
    size_t o_trow = tmp.add(trow), o_rowtab = tmp.add(rowtab), o_rowdst = tmp.add(rowdst), o_nrows = tmp.add(nrows);
    char* dres = nullptr;
    int rc = arena_upload(c, res, &dres, st);
    if (rc) return rc;
    void* dtmp = nullptr;
    MFDN_CUDA(c, cudaMalloc(&dtmp, tmp.buf.size()));
    MFDN_CUDA(c, cudaMemcpyAsync(dtmp, tmp.buf.data(), tmp.buf.size(), cudaMemcpyHostToDevice, st));
    const double* dvals = nullptr;
    void* vtmp = nullptr;
    rc = stage_values(c, values, values_on_device, n_values, st, &dvals, &vtmp);
    if (rc) { cudaFree(dtmp); return rc; }
    void* dslab = nullptr;
    cudaError_t e = cudaMalloc(&dslab, std::max<uint64_t>(cells, 1) * 16 + 256);
    void* ddtab = nullptr;
    // slack: in a mis-ordered MFDN_PRESORTED stream a record may meet the tables of another tuple and index up to
    // MAX_STATES3 * 32 doubles past its block
    if (e == cudaSuccess) e = cudaMalloc(&ddtab, (dtab_len + 32 * (uint64_t)MAX_STATES3) * sizeof(double));
    void* dvw = nullptr;
    if (e == cudaSuccess) e = cudaMalloc(&dvw, std::max<uint64_t>(vwcells, 1) * 16 + 256);        // slack: bulk copies are rounded up to 16 bytes
    if (e != cudaSuccess) {
        cudaFree(dtmp);
        if (vtmp) cudaFree(vtmp);
        if (dslab) cudaFree(dslab);
        if (ddtab) cudaFree(ddtab);
        return cuda_fail(c, e, "cudaMalloc(slab3/dtab3/vw20)");
    }
    c->owned.push_back(dslab);
    c->owned.push_back(ddtab);
    c->owned.push_back(dvw);
    Retile3 p;
    p.n_tup = nt;
    p.tdesc = (const int4*)((char*)dtmp + o_desc);
    p.sgrp = (const uint4*)(dres + o_sgrp);
    p.rowmap = (const int32_t*)((char*)dtmp + o_rm);
    p.chan_of = (const int32_t*)((char*)dtmp + o_cof);
    p.chan_off = (const int64_t*)((char*)dtmp + o_coff);
    p.chan_dim = (const int32_t*)((char*)dtmp + o_cdim);
    p.values = dvals;
    p.slab = (double*)dslab;
    long long groups = (long long)nt * nt;
    k_retile3<<<(unsigned)std::min<long long>(groups, 1 << 20), 64, 0, st>>>(p);
    k_vw20<<<(unsigned)std::min<long long>(groups, 1 << 20), 128, 0, st>>>(groups, p.sgrp, (const double*)dslab, c->t.wbin3, (uint32_t*)dvw, f32);
    Dtab3 q;
    q.tdesc = p.tdesc;
    q.tk = (const int4*)(dres + o_tk);
    q.trow = (const int2*)((char*)dtmp + o_trow);
    q.rowtab = (const int2*)((char*)dtmp + o_rowtab);
    q.rowdst = (const int2*)((char*)dtmp + o_rowdst);
    q.nrows = (const int32_t*)((char*)dtmp + o_nrows);
    q.sig = (const uint16_t*)(dres + o_sig);
    q.sigoff = (const int32_t*)(dres + o_sigoff);
    q.cg1 = c->t.cg1;
    q.cg1_off = c->t.cg1_off;
    q.cg2g = c->t.cg2g;
    q.nj = c->t.nj;
    q.dtab = (double*)ddtab;
    k_dtab3<<<(unsigned)nt, 256, 0, st>>>(q);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(dtmp);
    if (vtmp) cudaFree(vtmp);
    if (e != cudaSuccess) return cuda_fail(c, e, "k_retile3/k_dtab3");
    c->t.n_tup3 = nt;
    c->t.e3max = e3max;
    c->t.tuple_id3 = (const int32_t*)(dres + o_tid);
    c->t.tdesc3 = (const int4*)(dres + o_desc_rt);
    c->t.sgrp3 = p.sgrp;
    c->t.gbase3 = (const uint32_t*)(dres + o_gbase);
    c->t.n_buckets3 = (uint32_t)buckets;
    c->t.rowbase3 = (const uint32_t*)(dres + o_rowbase);
    c->t.colcum3 = (const uint16_t*)(dres + o_colcum);
    c->t.ncls3 = ncls;
    c->t.sig_len3 = (int)sig.size();
    c->t.stmask_len3 = (int)stmask.size();
    c->t.vw20 = (const uint32_t*)dvw;
    c->t.vw_f32 = f32;
    c->vw_bytes3 = (int64_t)(vwcells * 16);
    c->t.ab3 = ab_dense ? (const int2*)(dres + o_ab) : nullptr;
    c->t.slab3 = (const double*)dslab;
    c->t.stmask3 = (const unsigned long long*)(dres + o_sm);
    c->t.stm12_3 = (const unsigned long long*)(dres + o_sm12);
    c->t.stm12_off3 = (const int32_t*)(dres + o_sm12off);
    c->t.stm12_len3 = (int)stm12.size();
    c->t.tk3 = q.tk;
    c->t.jinfo3 = (const int2*)(dres + o_jinfo);
    c->t.dtab3 = (const double*)ddtab;
    c->t.sig3 = q.sig;
    c->t.mstart3 = (const uint16_t*)(dres + o_mstart);
    c->t.mstoff3 = (const int32_t*)(dres + o_mstoff);
    c->t.isig3 = (const uint16_t*)(dres + o_isig);
    c->t.torb3 = (const int4*)(dres + o_torb);
    c->t.spsidx3 = (const int32_t*)(dres + o_spsidx);
    c->h_tuple_id3 = tuple_id;
    c->h_tdesc3 = tdesc_rt;
    c->h_mstart3 = mstart;
    c->h_mstoff3 = mstoff;
    c->h_sgrp3 = sgrp;
    c->slab_bytes3 = (int64_t)(cells * 16);
    c->dtab_bytes3 = (int64_t)(dtab_len * sizeof(double));
    c->has3 = true;
    return MFDN_OK;
}

extern "C" int mfdn_coupled_upload_2b(mfdn_ctx* c, int32_t n_chan, const int32_t* chan_J, const int32_t* chan_T,
                                      const int32_t* chan_par, const int32_t* chan_dim, const int64_t* chan_off,
                                      const int32_t* state_a, const int32_t* state_b, const double* values,
                                      int values_on_device, void* stream)
{
    if (!c) return MFDN_ERR_ARG;
    if (c->stage < 2) return fail(c, MFDN_ERR_STATE, "mfdn_coupled_upload_2b before mfdn_cg_build");
    if (c->has2) return fail(c, MFDN_ERR_STATE, "2-body table already uploaded");
    if (n_chan <= 0 || !chan_J || !chan_T || !chan_par || !chan_dim || !chan_off || !state_a || !state_b || !values)
        return fail(c, MFDN_ERR_ARG, "null or empty argument");
    cudaStream_t st = (cudaStream_t)stream;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    const int No = c->t.n_orb;
    const auto& tj = c->orb_twoj;
    std::vector<int32_t> chan_of(32 * 4, -1);
    int64_t n_states = 0, n_values = 0;
    for (int ch = 0; ch < n_chan; ch++) {
        int J = chan_J[ch], T = chan_T[ch], P = chan_par[ch];
        if (J < 0 || J > MAX_TWOJ || (T != 0 && T != 1) || (P != 0 && P != 1) || chan_dim[ch] < 0 || chan_off[ch] < 0)
            return fail(c, MFDN_ERR_TABLE, "bad channel quantum numbers");
        int32_t& slot = chan_of[J * 4 + T * 2 + P];
        if (slot >= 0) return fail(c, MFDN_ERR_TABLE, "duplicate channel");
        slot = ch;
        n_states += chan_dim[ch];
        n_values = std::max<int64_t>(n_values, chan_off[ch] + (int64_t)chan_dim[ch] * chan_dim[ch]);
    }
    std::vector<int64_t> tkeys;
    tkeys.reserve(n_states);
    {
        int64_t s = 0;
        for (int ch = 0; ch < n_chan; ch++)
            for (int r = 0; r < chan_dim[ch]; r++, s++) {
                int a = state_a[s], b = state_b[s];
                if (a < 0 || a > b || b >= No) return fail(c, MFDN_ERR_TABLE, "state orbitals not a<=b in range");
                if (((c->orb_l[a] + c->orb_l[b]) & 1) != chan_par[ch]) return fail(c, MFDN_ERR_TABLE, "state parity != channel parity");
                if (2 * chan_J[ch] < std::abs(tj[a] - tj[b]) || 2 * chan_J[ch] > tj[a] + tj[b]) return fail(c, MFDN_ERR_TABLE, "J triangle");
                if (a == b && !((chan_J[ch] + chan_T[ch]) & 1)) return fail(c, MFDN_ERR_TABLE, "a==b needs J+T odd");
                tkeys.push_back((int64_t)a * No + b);
            }
    }
    std::vector<int64_t> tuples = tkeys;
    std::sort(tuples.begin(), tuples.end());
    tuples.erase(std::unique(tuples.begin(), tuples.end()), tuples.end());
    const int nt = (int)tuples.size();
    if (nt == 0) return fail(c, MFDN_ERR_TABLE, "empty table");
    std::vector<int32_t> tuple_id((size_t)No * No, -1), rowmap_off(nt);
    std::vector<int4> tdesc(nt);
    size_t rm_size = 0;
    for (int t = 0; t < nt; t++) {
        int a = (int)(tuples[t] / No), b = (int)(tuples[t] % No);
        tuple_id[tuples[t]] = t;
        int Jmin = std::abs(tj[a] - tj[b]) / 2, Jmax = (tj[a] + tj[b]) / 2;
        int par = (c->orb_l[a] + c->orb_l[b]) & 1;
        tdesc[t].x = tj[a] | (tj[b] << 8) | ((a == b) << 24) | (par << 25);
        tdesc[t].y = Jmin | (Jmax << 8);
        tdesc[t].z = tdesc[t].w = 0;
        rowmap_off[t] = (int32_t)rm_size;
        rm_size += (size_t)(Jmax - Jmin + 1) * 2;
    }
    std::vector<int32_t> rowmap(rm_size, -1);
    {
        int64_t s = 0;
        for (int ch = 0; ch < n_chan; ch++)
            for (int r = 0; r < chan_dim[ch]; r++, s++) {
                int t = tuple_id[tkeys[s]];
                int32_t& slot = rowmap[rowmap_off[t] + (chan_J[ch] - (tdesc[t].y & 255)) * 2 + chan_T[ch]];
                if (slot >= 0) return fail(c, MFDN_ERR_TABLE, "duplicate state in channel");
                slot = r;
                unsigned long long m = ((unsigned long long)(uint32_t)tdesc[t].z) | ((unsigned long long)(uint32_t)tdesc[t].w << 32);
                m |= 1ull << (chan_J[ch] * 2 + chan_T[ch]);
                tdesc[t].z = (int)(uint32_t)(m & 0xFFFFFFFFu);
                tdesc[t].w = (int)(uint32_t)(m >> 32);
            }
    }
    std::vector<uint32_t> slab_off((size_t)nt * nt, NO_SLAB);
    uint64_t cells = 0;
    for (int tb = 0; tb < nt; tb++)
        for (int tk = 0; tk < nt; tk++) {
            int4 db = tdesc[tb], dk = tdesc[tk];
            if (((db.x ^ dk.x) >> 25) & 1) continue;
            int Jlo = std::max(db.y & 255, dk.y & 255), Jhi = std::min((db.y >> 8) & 255, (dk.y >> 8) & 255);
            if (Jhi < Jlo) continue;
            if (cells + (Jhi - Jlo + 1) >= 0xFFFFFFF0ull) return fail(c, MFDN_ERR_OOM, "table too large for 32-bit cell offsets");
            slab_off[(size_t)tb * nt + tk] = (uint32_t)cells;
            cells += Jhi - Jlo + 1;
        }
    Arena res, tmp;
    size_t o_tid = res.add(tuple_id), o_desc = res.add(tdesc), o_soff = res.add(slab_off);
    std::vector<int64_t> coff(chan_off, chan_off + n_chan);
    std::vector<int32_t> cdim(chan_dim, chan_dim + n_chan);
    size_t o_rm = tmp.add(rowmap), o_rmo = tmp.add(rowmap_off), o_cof = tmp.add(chan_of), o_coff = tmp.add(coff), o_cdim = tmp.add(cdim);
    char* dres = nullptr;
    int rc = arena_upload(c, res, &dres, st);
    if (rc) return rc;
    void* dtmp = nullptr;
    MFDN_CUDA(c, cudaMalloc(&dtmp, tmp.buf.size()));
    MFDN_CUDA(c, cudaMemcpyAsync(dtmp, tmp.buf.data(), tmp.buf.size(), cudaMemcpyHostToDevice, st));
    const double* dvals = nullptr;
    void* vtmp = nullptr;
    rc = stage_values(c, values, values_on_device, n_values, st, &dvals, &vtmp);
    if (rc) { cudaFree(dtmp); return rc; }
    void* dslab = nullptr;
    cudaError_t e = cudaMalloc(&dslab, std::max<uint64_t>(cells, 1) * CELL2 * sizeof(double));
    if (e != cudaSuccess) { cudaFree(dtmp); if (vtmp) cudaFree(vtmp); return cuda_fail(c, e, "cudaMalloc(slab2)"); }
    c->owned.push_back(dslab);
    Retile2 p;
    p.n_tup = nt;
    p.tdesc = (const int4*)(dres + o_desc);
    p.slab_off = (const uint32_t*)(dres + o_soff);
    p.rowmap = (const int32_t*)((char*)dtmp + o_rm);
    p.rowmap_off = (const int32_t*)((char*)dtmp + o_rmo);
    p.chan_of = (const int32_t*)((char*)dtmp + o_cof);
    p.chan_off = (const int64_t*)((char*)dtmp + o_coff);
    p.chan_dim = (const int32_t*)((char*)dtmp + o_cdim);
    p.values = dvals;
    p.slab = (double*)dslab;
    long long groups = (long long)nt * nt;
    k_retile2<<<(unsigned)std::min<long long>((groups + 127) / 128, 1 << 16), 128, 0, st>>>(p);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(dtmp);
    if (vtmp) cudaFree(vtmp);
    if (e != cudaSuccess) return cuda_fail(c, e, "k_retile2");
    c->t.n_tup2 = nt;
    c->t.tuple_id2 = (const int32_t*)(dres + o_tid);
    c->t.tdesc2 = p.tdesc;
    c->t.slab_off2 = p.slab_off;
    c->t.slab2 = (const double*)dslab;
    c->slab_bytes2 = (int64_t)(cells * CELL2 * sizeof(double));
    c->has2 = true;
    return MFDN_OK;
}

// ------------------------------------------------------------------------------------------ misc
extern "C" int64_t mfdn_bad_request_count(mfdn_ctx* c, void* stream)
{
    if (!c || c->stage < 1) return -1;
    unsigned long long v = 0;
    cudaSetDevice(c->device);
    if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return -1;
    if (cudaMemcpy(&v, c->t.bad_count, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return (int64_t)v;
}

extern "C" int64_t mfdn_info(mfdn_ctx* c, int which)
{
    if (!c) return -1;
    switch (which) {
        case 0: return c->t.n_tup2;
        case 1: return c->t.n_tup3;
        case 2: return c->slab_bytes2;
        case 3: return c->slab_bytes3;
        case 4: return c->n_cg1;
        case 5: return c->n_cg2;
        case 6: return c->launches.load();
        case 7: return c->dtab_bytes3;
        case 8: return c->vw_bytes3;
        case 9: return c->t.n_buckets3;
        default: return -1;
    }
}

extern "C" const char* mfdn_last_error(mfdn_ctx* c)
{
    if (!c) return "null context";
    static thread_local std::string copy;   // valid until the calling thread's next mfdn_last_error
    std::lock_guard<std::mutex> lk(c->mu);
    copy = c->err;
    return copy.c_str();
}

extern "C" void mfdn_destroy(mfdn_ctx* c)
{
    if (!c) return;
    cudaSetDevice(c->device);
    for (void* p : c->owned) cudaFree(p);
    for (auto& ev : c->ev_pending) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); cudaEventDestroy(ev.d); cudaEventDestroy(ev.c); }
    for (auto e : c->ev_pool) cudaEventDestroy(e);
    for (auto s : c->hs) if (s) cudaStreamDestroy(s);
    delete c;
}
