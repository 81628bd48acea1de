// ozfft.cu -- plan, stage scheduling and the C ABI of include/ozfft.h.
// Axis passes z, y, x; each axis is one stage (n <= 32) or two stages with the twiddle
// fused into the second-stage matrices (Eq. 6).  The array between stages is
// fp64 (one correctly rounded pack per stage output, Alg. 2 line 16).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <set>
#include <string>
#include <vector>

#include "ozfft.h"
#include "stage.cuh"
#include "stage_simt.cuh"
#include "stage_tc.cuh"
#include "stage_bf.cuh"
#include "stage_f8.cuh"
#include "tables.cuh"
#include "probe.cuh"

using namespace oz;

namespace {

thread_local std::string g_err = "";
void set_err(const std::string &s) { g_err = s; }
bool cuda_ok(cudaError_t e, const char *what) {
    if (e == cudaSuccess) return true;
    set_err(std::string(what) + ": " + cudaGetErrorString(e));
    return false;
}

const Twiddles &twiddles() {
    static Twiddles T;
    static std::once_flag once;
    std::call_once(once, [] { build_twiddles(T); });
    return T;
}

// live plans: a destroyed (or never created) handle is recognised without touching freed memory
std::mutex g_plans_mu;
std::set<const void *> g_plans;

struct StageLaunch {
    StageGeom g;
    const ushort2 *mat_simt;  // [nmat][12][K][K] (a_R, a_I) canonical residues
    const uint8_t *mat_tc;    // digit planes for the tensor-core kernel (stage_tc.cuh)
    const uint8_t *mat_bf;    // matrix byte planes of the byte-fed kernel (stage_bf.cuh)
    const uint8_t *mat_f8;    // E4M3 hex-digit planes of the FP8 rung (stage_f8.cuh)
    const void *ctab_bf;      // its offset constants [nmat][K] x 16 B
    int axis;
    bool fused;               // byte-fed kernel, axis of length 1024: both stages in one launch (stage_bf.cuh BfFuse); g = first stage
    BfFuse fuse;              // second stage and group layout (ring and counters are filled in at launch from the plan)
};

}  // namespace

struct ozfft_plan_s {
    uint32_t magic;
    int nx, ny, nz, sign;
    long long count;
    int variant;  // 0 simt, 1 tensor-core (residue digits), 2 byte-fed tensor-core (default), 3 / 4 ablations on the simt kernel, 5 FP8 rung
    int sms;      // SM count of the plan's device
    int tc_per_sm[3];  // resident CTAs per SM of the residue-digit kernel instantiations (per device)
    const void *pa_bf;  // Phase-A constant matrix of the byte-fed kernel
    std::vector<StageLaunch> stages;
    std::vector<StageLaunch> stages_nat;  // the same passes with every intermediate array in natural order (ozfft_exec_axis)
    std::vector<void *> dev_allocs;
    size_t dev_bytes;
    DevConsts *d_consts;
    void *work;
    void *ring;           // fused axes: Y' ring (L2 resident) and the group counters
    unsigned int *ctr;
    int ring_slots, fuse_lag, max_groups;
    bool fuse;            // schedule: fused axes where the shape allows (OZFFT_SCHEDULE=unfused turns it off)
    void *h_in, *h_out;  // device staging for ozfft_exec_host (lazy)
    bool pipelined;      // exec_host overlaps the copies with the passes
    std::vector<StageLaunch> slab_stages;  // z and y stages of one slab of nx/PIPE planes
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_in[8], ev_out[8], ev_start;
};

namespace {

constexpr uint32_t PLAN_MAGIC = 0x4F5A4646u;
constexpr int PIPE = 8;  // slabs / chunks of the host-buffer pipeline

bool is_pow2(int n) { return n >= 2 && (n & (n - 1)) == 0; }

void fill_consts(DevConsts &c) {
    CrtConsts C;
    build_crt(C);
    for (int k = 0; k < R_MOD; k++) {
        const uint32_t m = (uint32_t)kModuli[k];
        c.m[k] = m;
        c.mu[k] = (uint32_t)((1ull << 32) / m);
        c.c16[k] = (uint32_t)((1ull << 16) % m);
        c.c32[k] = (uint32_t)((1ull << 32) % m);
        c.c48[k] = (uint32_t)((1ull << 48) % m);
        c.off28[k] = (uint32_t)((((1u << 28) + m - 1) / m) * m);
        c.offtc[k] = (uint32_t)((((1u << 25) + m - 1) / m) * m);
        for (int l = 0; l < 4; l++) c.u[k][l] = (uint32_t)(C.u[k] >> (32 * l));
        c.wlo[k] = (uint32_t)C.w[k];
        c.whi[k] = (uint32_t)(C.w[k] >> 32);
    }
    for (int k = 0; k < R_MOD; k++) {
        const uint32_t m = (uint32_t)kModuli[k];
        c.c18[k] = (uint32_t)((1ull << 18) % m);
        c.c36[k] = (uint32_t)((1ull << 36) % m);
        c.m2[k] = 2 * m;
        c.m2m2[k] = 2 * m * 0x10001u;
        c.off30[k] = (uint32_t)((((1u << 30) + m - 1) / m) * m);
    }
    {  // zC = round(2^149 / M) by binary long division
        u128 rem = 1;
        uint64_t q = 0;
        for (int b = 0; b < 149; b++) {
            rem <<= 1;
            q <<= 1;
            if (rem >= C.M) { rem -= C.M; q |= 1; }
        }
        if (rem * 2 >= C.M) q++;
        c.zC = (uint32_t)q;
    }
    {  // Phase-A matrix, two-limb shifted-column form: residue v = v0 + 256 v1 sits in operand bytes (2k, 2k+1);
       // row s holds byte s of u_k against v0 and byte s-1 against v1.  Operand order [chunk][row][16 B].
        uint8_t *pa = (uint8_t *)c.phaseA;
        memset(pa, 0, 512);
        for (int s = 0; s < 16; s++)
            for (int k = 0; k < R_MOD; k++)
                for (int l = 0; l < 2; l++) {
                    const int sh = s - l, kap = 2 * k + l;
                    const uint8_t b = sh < 0 ? 0 : (uint8_t)(C.u[k] >> (8 * sh));
                    pa[(kap / 16) * 256 + s * 16 + kap % 16] = b;
                }
    }
    for (int k = 0; k < R_MOD; k++) {  // ablation tables: Garner mixed-radix constants, idempotent byte slices
        const int mk = kModuli[k];
        long prod = 1 % mk;
        for (int j = 0; j < R_MOD; j++) {
            c.gprod[j][k] = (uint16_t)prod;  // product of the first j moduli, mod m_k
            if (j == k) c.ginv[k] = (uint16_t)mod_inverse((int)prod, mk);
            prod = (prod * (kModuli[j] % mk)) % mk;
        }
        for (int s = 0; s < 16; s++) c.uslice[k][s] = (uint8_t)(C.u[k] >> (8 * s));
    }
    for (int l = 0; l < 4; l++) {
        c.M[l] = (uint32_t)(C.M >> (32 * l));
        c.Mh[l] = (uint32_t)(C.Mhalf >> (32 * l));
    }
}

// table index t (into omega_1024) of matrix `mid`, row k, column j.  fusedN == 0: plain F_K;
// else the twiddle-fused second-stage matrix of a length-fusedN transform for k2 = mid (Eq. 6).
inline int tw_index(int K, int fusedN, int mid, int k, int j) {
    if (!fusedN) return (int)(((long)(TABLE_N / K) * j * k) % TABLE_N);
    return (int)(((long)(TABLE_N / fusedN) * j * (mid + 32L * k)) % TABLE_N);
}

struct MatKey {
    int K, fusedN;
    bool operator<(const MatKey &o) const { return K != o.K ? K < o.K : fusedN < o.fusedN; }
};
struct MatSet {
    const ushort2 *simt;
    const uint8_t *tc, *bf, *f8;
    const void *ctab;
};
typedef std::map<MatKey, MatSet> MatMap;

void *dev_upload(ozfft_plan_s *p, const void *src, size_t bytes) {
    void *d = nullptr;
    if (!cuda_ok(cudaMalloc(&d, bytes), "cudaMalloc(table)")) return nullptr;
    if (!cuda_ok(cudaMemcpy(d, src, bytes, cudaMemcpyHostToDevice), "cudaMemcpy(table)")) { cudaFree(d); return nullptr; }
    p->dev_allocs.push_back(d);
    p->dev_bytes += bytes;
    return d;
}

const ushort2 *build_mat_simt(ozfft_plan_s *p, int K, int fusedN) {
    const Twiddles &T = twiddles();
    const int nmat = fusedN ? 32 : 1;
    std::vector<ushort2> h((size_t)nmat * 12 * K * K);
    for (int mid = 0; mid < nmat; mid++)
        for (int i = 0; i < 12; i++)
            for (int k = 0; k < K; k++)
                for (int j = 0; j < K; j++) {
                    const int t = tw_index(K, fusedN, mid, k, j);
                    ushort2 a;
                    a.x = (unsigned short)residue_of(T.c[t], kModuli[i]);
                    a.y = (unsigned short)residue_of((int64_t)p->sign * T.s[t], kModuli[i]);
                    h[(((size_t)mid * 12 + i) * K + k) * K + j] = a;
                }
    return (const ushort2 *)dev_upload(p, h.data(), h.size() * sizeof(ushort2));
}

struct AxisDesc {
    bool contiguous;
    long long outer, N, inner;  // strided: element (o, i, z) at (o*N + i)*inner + z; contiguous: pencil P at P*N
};

// perm_out: the second stage of this (contiguous) axis writes index k1 + p k2 instead of k2 + 32 k1; unperm = p > 0: the first
// stage of this axis reads an inner index permuted that way and writes the natural one (StageGeom::patch)
bool add_axis(ozfft_plan_s *p, const AxisDesc &a, int axis, MatMap &mats, std::vector<StageLaunch> &dst, bool perm_out = false, int unperm = 0, bool fuse = false) {
    const int N = (int)a.N;
    const bool two = N > 32;
    const int q = two ? 32 : N, pp = two ? N / 32 : 1;
    auto get = [&](int K, int fusedN, StageLaunch &s) -> bool {
        MatKey key{K, fusedN};
        auto it = mats.find(key);
        if (it == mats.end()) {
            MatSet ms{};
            if (p->variant == 0 || p->variant == 3 || p->variant == 4) {
                ms.simt = build_mat_simt(p, K, fusedN);
                if (!ms.simt) return false;
            } else if (p->variant == 1) {
                std::vector<uint8_t> h;
                build_mat_tc(h, K, fusedN, p->sign, twiddles());
                ms.tc = (const uint8_t *)dev_upload(p, h.data(), h.size());
                if (!ms.tc) return false;
            } else if (p->variant == 5) {
                std::vector<uint8_t> h;
                build_mat_f8(h, K, fusedN, p->sign, twiddles());
                ms.f8 = (const uint8_t *)dev_upload(p, h.data(), h.size());
                if (!ms.f8) return false;
            } else {
                std::vector<uint8_t> h;
                std::vector<uint32_t> c;
                build_mat_bf(h, c, K, fusedN, p->sign, twiddles());
                ms.bf = (const uint8_t *)dev_upload(p, h.data(), h.size());
                ms.ctab = dev_upload(p, c.data(), c.size() * 4);
                if (!ms.bf || !ms.ctab) return false;
            }
            it = mats.insert({key, ms}).first;
        }
        s.mat_simt = it->second.simt;
        s.mat_tc = it->second.tc;
        s.mat_bf = it->second.bf;
        s.mat_f8 = it->second.f8;
        s.ctab_bf = it->second.ctab;
        return true;
    };
    StageLaunch s1{}, s2{};
    s1.axis = s2.axis = axis;
    StageGeom &g1 = s1.g, &g2 = s2.g;
    g1.K = q; g1.matsel = 0;
    g2.K = pp; g2.matsel = 1; g2.ns = 32;
    g1.ns = pp;
    if (!a.contiguous) {
        const long long I = a.inner;
        g1.nb = g2.nb = (int)((I + 31) / 32); g1.no = g2.no = (int)a.outer;
        g1.ncols = g2.ncols = (int)I;
        g1.ib = 32; g1.is = I; g1.io = a.N * I;
        g1.lane = 1; g1.ji = pp * I; g1.ko = pp * I; g1.order = 0;
        g2.ib = 32; g2.is = pp * I; g2.io = a.N * I;
        g2.ob = 32; g2.os = I; g2.oo = a.N * I;
        g2.lane = 1; g2.ji = I; g2.ko = 32 * I; g2.order = 0;
    } else {
        const long long Pn = a.outer;
        g1.nb = g2.nb = (int)((Pn + 31) / 32); g1.no = g2.no = 1;
        g1.ncols = g2.ncols = (int)Pn;
        g1.ib = 32 * a.N; g1.is = 1; g1.io = 0;
        g1.lane = a.N; g1.ji = pp; g1.ko = pp; g1.order = 1;
        if (two && pp == 32) {  // N = 1024: a block is one pencil, lanes along j1 (adjacent elements): coalesced
            g1.nb = (int)Pn; g1.ncols = 32 * (int)Pn; g1.ns = 1; g1.ib = a.N; g1.is = 0; g1.lane = 1; g1.order = 0;
        }
        g2.ib = 32 * a.N; g2.is = pp; g2.io = 0;
        g2.ob = 32 * a.N; g2.os = 1; g2.oo = 0;
        g2.lane = a.N; g2.ji = 1; g2.ko = 32; g2.order = 1;
    }
    g1.ob = g1.ib; g1.os = g1.is; g1.oo = g1.io;
    g1.olane = g1.lane; g2.olane = g2.lane;
    if (a.contiguous && two && pp == 32) {
        // N = 1024 on the contiguous axis: the array between the two stages is ours to lay out.  Y'[k2][pencil][j1]
        // (instead of the input's own positions) makes a second-stage tile -- 128 pencils that share k2 -- one
        // contiguous 64 KB read; the first stage still writes 512-byte runs (32 lanes along j1).
        const long long Pn = a.outer;
        g1.ob = 32; g1.ko = Pn * 32;
        g2.ib = 32 * 32; g2.lane = 32; g2.ji = 1; g2.is = Pn * 32;
    }
    if (perm_out) { g2.os = pp; g2.ko = 1; }
    for (StageGeom *gp : {&g1, &g2}) {  // column addressing of the byte-fed kernel: four blocks of 32 lanes
        gp->ci = StageGeom::ColMap{0, 0, 31, 5, 4 * gp->ib, 0, gp->lane, gp->ib};
        gp->co = StageGeom::ColMap{0, 0, 31, 5, 4 * gp->ob, 0, gp->olane, gp->ob};
    }
    if (unperm) {  // 8 (k1) x 16 (k2) patch: permuted index k1 + p k2 in, natural index k2 + 32 k1 out
        g1.ci = StageGeom::ColMap{1, 1, 7, 3, 8, 16LL * unperm, 1, unperm};
        g1.co = StageGeom::ColMap{1, 1, 7, 3, 256, 16, 32, 1};
    }
    if (!get(q, 0, s1)) return false;
    const long long cols = a.contiguous ? a.outer : a.inner;  // columns along the b coordinate
    if (fuse && p->variant == 2 && two && pp == 32 && cols % 128 == 0) {
        // fused axis: Y' of a group of 128 pencils (32 x 4096 elements) lives in a ring slot, laid out [k2][j1 or pencil][...]
        if (!get(pp, N, s2)) return false;
        StageLaunch sf = s1;
        sf.fused = true;
        BfFuse &f = sf.fuse;
        f = BfFuse{};
        f.g2 = g2;
        f.mat2 = s2.mat_bf;
        f.ctab2 = (const uint4 *)s2.ctab_bf;
        if (unperm) f.g2.co = g1.co;  // the group's 128 columns are the 8 x 16 patch: the second stage stores them at their natural places
        sf.g.os = 0; sf.g.oo = 0; sf.g.ko = 4096;
        f.g2.is = 4096; f.g2.io = 0;
        if (a.contiguous) {
            // first-stage tile = 4 pencils x 32 j1; second-stage column = pencil.  Ring [k2][j1][pencil]: the second stage's loads
            // are coalesced across its columns like on the strided axes (its latency-bound side); the first stage pays with
            // 16-byte stores 2 KB apart, which stay in L2
            sf.g.co = StageGeom::ColMap{0, 0, 31, 5, 4, 0, 128, 1};
            f.g2.ci = StageGeom::ColMap{0, 0, 127, 7, 0, 0, 1, 0};
            f.g2.ji = 128;
            f.G = (int)(cols / 128);
            f.lg_nbt = 30;
            f.s1_mulb = 32; f.s1_tlb = 1; f.s1_tls = 0; f.r1_tlb = 1; f.r1_tls = 0;
        } else {             // first-stage tile = one j1 of 128 lanes -> ring [k2][j1][lane]
            sf.g.co = StageGeom::ColMap{0, 0, 127, 7, 0, 0, 1, 0};
            sf.g.os = 128;
            f.g2.ci = StageGeom::ColMap{0, 0, 127, 7, 0, 0, 1, 0};
            f.g2.ji = 128;
            const int nbt = (int)(cols / 128);
            f.G = nbt * (int)a.outer;
            f.lg_nbt = 0;
            while ((1 << f.lg_nbt) < nbt) f.lg_nbt++;
            f.s1_mulb = 1; f.s1_tlb = 0; f.s1_tls = 1; f.r1_tlb = 0; f.r1_tls = 1;
        }
        if (f.G > p->max_groups) p->max_groups = f.G;
        dst.push_back(sf);
        return true;
    }
    dst.push_back(s1);
    if (two) {
        if (!get(pp, N, s2)) return false;
        dst.push_back(s2);
    }
    return true;
}

int pick_variant() {
    const char *v = getenv("OZFFT_VARIANT");
    if (v && !strcmp(v, "simt")) return 0;
    if (v && !strcmp(v, "tc")) return 1;
    if (v && !strcmp(v, "garner")) return 3;   // ablation: SIMT kernel with recursive Garner reconstruction
    if (v && !strcmp(v, "fp64sum")) return 4;
    if (v && !strcmp(v, "fp8")) return 5;      // measured rung: kind::f8f6f4 E4M3 digit planes + residue-domain Karatsuba  // ablation: SIMT kernel with the naive fp64 Phase B (NOT exact, uses fp64)
    return 2;
}

ozfft_plan_s *make_plan(int nx, int ny, int nz, int sign, bool batched1d) {
    if (sign != -1 && sign != 1) { set_err("sign must be -1 (forward) or +1 (inverse)"); return nullptr; }
    int dev = 0;
    cudaDeviceProp prop;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice") || !cuda_ok(cudaGetDeviceProperties(&prop, dev), "cudaGetDeviceProperties"))
        return nullptr;
    if (prop.major != 10) { set_err("ozfft needs an sm_100 device (B200); no fallback path exists"); return nullptr; }
    ozfft_plan_s *p = new ozfft_plan_s();
    p->magic = PLAN_MAGIC;
    p->nx = nx; p->ny = ny; p->nz = nz; p->sign = sign;
    p->count = (long long)nx * ny * nz;
    p->variant = pick_variant();
    p->dev_bytes = 0;
    p->work = p->h_in = p->h_out = nullptr;
    p->ring = nullptr; p->ctr = nullptr; p->max_groups = 0;
    {   // schedule of the byte-fed kernel: axes of length 1024 run both stages in one launch unless OZFFT_SCHEDULE=unfused
        const char *sch = getenv("OZFFT_SCHEDULE");
        p->fuse = !(sch && !strcmp(sch, "unfused"));
        // lag 8 groups, ring 16 slots = 32 MB (a power of two: the slot index is a mask; measured at 1024^3: lag 3 / 4 / 6 / 8 / 12 -> 191 / 144 / 131 / 130 / 132 ms: below ~6 the
        // second-stage tiles catch up with the first-stage tiles still in flight on the 148 SMs and wait)
        p->fuse_lag = 8;
        p->ring_slots = 16;
    }
    p->pipelined = false;
    p->s_in = p->s_out = nullptr;
    DevConsts hc;
    fill_consts(hc);
    p->d_consts = (DevConsts *)dev_upload(p, &hc, sizeof(hc));
    MatMap mats;
    bool ok = p->d_consts != nullptr;
    p->sms = prop.multiProcessorCount;
    p->pa_bf = nullptr;
    if (ok && p->variant == 2) {
        CrtConsts C;
        build_crt(C);
        std::vector<uint8_t> pa(BF_PA_BYTES);
        build_pa_bf(pa.data(), C);
        p->pa_bf = dev_upload(p, pa.data(), pa.size());
        ok = p->pa_bf != nullptr;
    }
    if (batched1d) {  // nx = batch, nz = n
        ok = ok && add_axis(p, AxisDesc{true, nx, nz, 1}, 0, mats, p->stages, false, 0, p->fuse);
        if (ok && !p->stages.empty() && p->stages[0].fused) ok = add_axis(p, AxisDesc{true, nx, nz, 1}, 0, mats, p->stages_nat);
    } else {
        // byte-fed kernel, nz = 1024: the z pass leaves its output permuted along z and the first y stage undoes it (stage.cuh).
        // Measured at nz = 512: the patch costs the y stage 0.5 ms and the z pass gains nothing (it is bound by its lane-per-pencil
        // loads there, not by the partial sectors), so shorter z axes keep the natural order.
        const bool perm = p->variant == 2 && nz == 1024;
        ok = ok && add_axis(p, AxisDesc{true, (long long)nx * ny, nz, 1}, 0, mats, p->stages, perm, 0, p->fuse);
        ok = ok && add_axis(p, AxisDesc{false, nx, ny, nz}, 1, mats, p->stages, false, perm ? nz / 32 : 0, p->fuse);
        ok = ok && add_axis(p, AxisDesc{false, 1, nx, (long long)ny * nz}, 2, mats, p->stages, false, 0, p->fuse);
        bool any_fused = false;
        for (const StageLaunch &sl : p->stages) any_fused = any_fused || sl.fused;
        if (perm || any_fused) {
            ok = ok && add_axis(p, AxisDesc{true, (long long)nx * ny, nz, 1}, 0, mats, p->stages_nat);
            ok = ok && add_axis(p, AxisDesc{false, nx, ny, nz}, 1, mats, p->stages_nat);
            ok = ok && add_axis(p, AxisDesc{false, 1, nx, (long long)ny * nz}, 2, mats, p->stages_nat);
        }
        // host-buffer pipeline (ozfft_exec_host): the z and y passes run per slab of nx/8 planes as the slabs arrive,
        // the x pass per chunk of ny/8 rows whose results leave while the next chunk computes
        const int xs = nx / PIPE, yc = ny / PIPE;
        if (ok && nx >= PIPE && ny >= PIPE && p->count >= (1ll << 24) && ((long long)xs * ny) % 64 == 0 && ((long long)yc * nz) % 64 == 0) {
            ok = ok && add_axis(p, AxisDesc{true, (long long)xs * ny, nz, 1}, 0, mats, p->slab_stages, perm, 0);
            ok = ok && add_axis(p, AxisDesc{false, xs, ny, nz}, 1, mats, p->slab_stages, false, perm ? nz / 32 : 0);
            p->pipelined = ok;
        }
    }
    if (ok) {
        ok = cuda_ok(cudaMalloc(&p->work, (size_t)p->count * 16), "cudaMalloc(workspace)");
        if (ok) p->dev_bytes += (size_t)p->count * 16;
    }
    if (ok && p->max_groups) {  // fused axes: the Y' ring and two counters per group
        const size_t rb = (size_t)p->ring_slots * BF_GROUP_ELEMS * 16, cb = (size_t)p->max_groups * 8;
        ok = cuda_ok(cudaMalloc(&p->ring, rb), "cudaMalloc(ring)") && cuda_ok(cudaMalloc((void **)&p->ctr, cb), "cudaMalloc(counters)");
        if (ok) p->dev_bytes += rb + cb;
    }
    // per plan, on the plan's device: kernel attributes and the constant bank (both are per-device state)
    if (ok && (p->variant == 0 || p->variant == 3 || p->variant == 4)) {
        const int sm = 32 * 32 * 16 + 12 * 32 * 32 * 4;
        ok = cuda_ok(cudaFuncSetAttribute(stage_simt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, sm), "cudaFuncSetAttribute") &&
             cuda_ok(cudaFuncSetAttribute(stage_garner_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, sm), "cudaFuncSetAttribute") &&
             cuda_ok(cudaFuncSetAttribute(stage_fp64sum_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, sm), "cudaFuncSetAttribute");
    }
    if (ok && (p->variant == 1 || p->variant == 2 || p->variant == 5)) ok = stage_tc_prepare(hc);
    if (ok && p->variant == 5) ok = stage_f8_prepare();  // uploads the constant bank both tensor-core kernels read
    if (ok && p->variant == 1) stage_tc_occupancy(p->tc_per_sm);
    if (ok && p->variant == 2) ok = stage_bf_prepare();
    if (!ok && g_err.empty()) set_err("kernel attribute setup failed");
    {
        std::lock_guard<std::mutex> lk(g_plans_mu);
        g_plans.insert(p);
    }
    if (!ok) {
        std::string keep = g_err;
        ozfft_plan_destroy(p);
        set_err(keep);
        return nullptr;
    }
    return p;
}

bool valid(ozfft_plan p) {
    std::lock_guard<std::mutex> lk(g_plans_mu);
    return p && g_plans.count(p) != 0;
}

int launch_stage(ozfft_plan p, const StageLaunch &s, const void *src, void *dst, cudaStream_t st) {
    const long long nt = (long long)s.g.nb * s.g.ns * s.g.no;
    if (p->variant == 5) {
        return cuda_ok(stage_f8_launch(s.g, src, dst, s.mat_f8, p->sms, st), "stage_f8_kernel launch") ? OZFFT_OK : OZFFT_ECUDA;
    }
    if (p->variant == 2 && s.fused) {
        BfFuse f = s.fuse;
        f.ring = (uint4 *)p->ring;
        f.wr_done = p->ctr;
        f.rd_done = p->ctr + p->max_groups;
        f.Lg = p->fuse_lag < f.G ? p->fuse_lag : f.G;
        f.R = p->ring_slots;
        if (stage_bf_launch_fused(s.g, f, src, dst, s.mat_bf, s.ctab_bf, p->pa_bf, p->sms, st)) return OZFFT_OK;
        set_err(std::string("stage_bf_kernel (fused axis) launch: ") + cudaGetErrorString(cudaGetLastError()));
        return OZFFT_ECUDA;
    }
    if (p->variant == 2) {
        if (stage_bf_launch(s.g, src, dst, s.mat_bf, s.ctab_bf, p->pa_bf, p->sms, st)) return OZFFT_OK;
        set_err(std::string("stage_bf_kernel launch: ") + cudaGetErrorString(cudaGetLastError()));
        return OZFFT_ECUDA;
    }
    if (p->variant == 1) {
        if (stage_tc_launch(s.g, src, dst, s.mat_tc, p->sms, p->tc_per_sm, st)) return OZFFT_OK;
        set_err(std::string("stage_tc_kernel launch: ") + cudaGetErrorString(cudaGetLastError()));
        return OZFFT_ECUDA;
    }
    const size_t sm = (size_t)s.g.K * 32 * 16 + (size_t)12 * s.g.K * 32 * 4;
    if (p->variant == 3) stage_garner_kernel<<<(unsigned)nt, SIMT_THREADS, sm, st>>>(s.g, (const ulonglong2 *)src, (ulonglong2 *)dst, s.mat_simt, p->d_consts);
    else if (p->variant == 4) stage_fp64sum_kernel<<<(unsigned)nt, SIMT_THREADS, sm, st>>>(s.g, (const ulonglong2 *)src, (ulonglong2 *)dst, s.mat_simt, p->d_consts);
    else stage_simt_kernel<<<(unsigned)nt, SIMT_THREADS, sm, st>>>(s.g, (const ulonglong2 *)src, (ulonglong2 *)dst, s.mat_simt, p->d_consts);
    return cuda_ok(cudaGetLastError(), "stage_simt_kernel launch") ? OZFFT_OK : OZFFT_ECUDA;
}

// run stages [first, last) : src -> ... -> dst, alternating through the plan workspace so the last lands in dst
int run_stages(ozfft_plan p, const std::vector<StageLaunch> &stages, size_t first, size_t last, const void *in, void *out, cudaStream_t st) {
    const size_t L = last - first;
    const void *src = in;
    for (size_t i = 0; i < L; i++) {
        void *dst = ((L - 1 - i) & 1) ? p->work : out;
        int rc = launch_stage(p, stages[first + i], src, dst, st);
        if (rc) return rc;
        src = dst;
    }
    return OZFFT_OK;
}

bool check_ptrs(const void *in, void *out) {
    if (!in || !out || ((uintptr_t)in & 15) || ((uintptr_t)out & 15) || in == out) {
        set_err("in/out must be distinct, non-null, 16-byte aligned device pointers");
        return false;
    }
    return true;
}

}  // namespace

extern "C" {

ozfft_plan ozfft_plan_create(int nx, int ny, int nz, int sign) {
    if (!is_pow2(nx) || !is_pow2(ny) || !is_pow2(nz) || nx > 1024 || ny > 1024 || nz > 1024) {
        set_err("sizes must be powers of two in [2, 1024]");
        return nullptr;
    }
    return make_plan(nx, ny, nz, sign, false);
}

ozfft_plan ozfft_plan_create_1d(int n, int batch, int sign) {
    if (!is_pow2(n) || n > 1024 || batch < 1 || (long long)n * batch > (1ll << 30)) {
        set_err("n must be a power of two in [2, 1024], batch >= 1 and n * batch <= 2^30 elements");
        return nullptr;
    }
    return make_plan(batch, 1, n, sign, true);
}

int ozfft_exec(ozfft_plan p, const void *in, void *out, void *stream) {
    if (!valid(p)) { set_err("invalid or destroyed plan"); return OZFFT_EINVAL; }
    if (!check_ptrs(in, out)) return OZFFT_EINVAL;
    return run_stages(p, p->stages, 0, p->stages.size(), in, out, (cudaStream_t)stream);
}

int ozfft_exec_axis(ozfft_plan p, int axis, const void *in, void *out, void *stream) {
    if (!valid(p)) { set_err("invalid or destroyed plan"); return OZFFT_EINVAL; }
    if (!check_ptrs(in, out)) return OZFFT_EINVAL;
    const std::vector<StageLaunch> &sl = p->stages_nat.empty() ? p->stages : p->stages_nat;  // natural order in, natural order out
    size_t first = sl.size(), last = 0;
    for (size_t i = 0; i < sl.size(); i++)
        if (sl[i].axis == axis) { first = i < first ? i : first; last = i + 1; }
    if (first >= last) { set_err("no such axis in this plan"); return OZFFT_EINVAL; }
    return run_stages(p, sl, first, last, in, out, (cudaStream_t)stream);
}

// pipelined host-buffer transform of a 3-D plan: H2D slab s || z,y passes of slab s-1;  x pass of chunk c || D2H of chunk c-1
static int exec_host_pipelined_body(ozfft_plan p, const char *hin, char *hout, cudaStream_t st) {
    const long long nx = p->nx, ny = p->ny, nz = p->nz;
    const long long xs = nx / PIPE, yc = ny / PIPE;
    const size_t slab_elems = (size_t)(xs * ny * nz), slab_bytes = slab_elems * 16;
    if (!p->s_in) {
        if (!cuda_ok(cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking), "cudaStreamCreate") ||
            !cuda_ok(cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking), "cudaStreamCreate")) return OZFFT_ECUDA;
        for (int i = 0; i < PIPE; i++) {
            if (!cuda_ok(cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming), "cudaEventCreate") ||
                !cuda_ok(cudaEventCreateWithFlags(&p->ev_out[i], cudaEventDisableTiming), "cudaEventCreate")) return OZFFT_ECUDA;
        }
        if (!cuda_ok(cudaEventCreateWithFlags(&p->ev_start, cudaEventDisableTiming), "cudaEventCreate")) return OZFFT_ECUDA;
    }
    const std::vector<StageLaunch> &full = p->stages_nat.empty() ? p->stages : p->stages_nat;  // stage by stage (the x pass runs per chunk)
    const size_t L = full.size(), Lzy = p->slab_stages.size();
    auto buf_of = [&](size_t i) -> char * { return (char *)(((L - 1 - i) & 1) ? p->work : p->h_out); };  // as run_stages
    // copies start once earlier work on the caller's stream is done
    if (!cuda_ok(cudaEventRecord(p->ev_start, st), "cudaEventRecord") || !cuda_ok(cudaStreamWaitEvent(p->s_in, p->ev_start, 0), "cudaStreamWaitEvent") ||
        !cuda_ok(cudaStreamWaitEvent(p->s_out, p->ev_start, 0), "cudaStreamWaitEvent")) return OZFFT_ECUDA;
    for (int s = 0; s < PIPE; s++) {
        if (!cuda_ok(cudaMemcpyAsync((char *)p->h_in + s * slab_bytes, hin + s * slab_bytes, slab_bytes, cudaMemcpyHostToDevice, p->s_in), "H2D slab")) return OZFFT_ECUDA;
        if (!cuda_ok(cudaEventRecord(p->ev_in[s], p->s_in), "cudaEventRecord")) return OZFFT_ECUDA;
    }
    for (int s = 0; s < PIPE; s++) {  // z and y passes of slab s
        if (!cuda_ok(cudaStreamWaitEvent(st, p->ev_in[s], 0), "cudaStreamWaitEvent")) return OZFFT_ECUDA;
        const char *src = (const char *)p->h_in + s * slab_bytes;
        for (size_t i = 0; i < Lzy; i++) {
            char *dst = buf_of(i) + s * slab_bytes;
            int rc = launch_stage(p, p->slab_stages[i], src, dst, st);
            if (rc) return rc;
            src = dst;
        }
    }
    for (int c = 0; c < PIPE; c++) {  // x pass of the rows y in [c*yc, (c+1)*yc), then their way home
        const size_t off = (size_t)(c * yc * nz) * 16;
        const char *src = (Lzy ? buf_of(Lzy - 1) : (char *)p->h_in) + off;
        for (size_t i = Lzy; i < L; i++) {
            StageLaunch sl = full[i];
            sl.g.nb = (int)(yc * nz / 32);
            sl.g.ncols = (int)(yc * nz);
            char *dst = buf_of(i) + off;
            int rc = launch_stage(p, sl, src, dst, st);
            if (rc) return rc;
            src = dst;
        }
        if (!cuda_ok(cudaEventRecord(p->ev_out[c], st), "cudaEventRecord") || !cuda_ok(cudaStreamWaitEvent(p->s_out, p->ev_out[c], 0), "cudaStreamWaitEvent")) return OZFFT_ECUDA;
        if (!cuda_ok(cudaMemcpy2DAsync(hout + off, (size_t)(ny * nz) * 16, (char *)p->h_out + off, (size_t)(ny * nz) * 16,
                                       (size_t)(yc * nz) * 16, (size_t)nx, cudaMemcpyDeviceToHost, p->s_out), "D2H chunk")) return OZFFT_ECUDA;
    }
    if (!cuda_ok(cudaStreamSynchronize(p->s_out), "cudaStreamSynchronize")) return OZFFT_ECUDA;
    return cuda_ok(cudaStreamSynchronize(st), "cudaStreamSynchronize") ? OZFFT_OK : OZFFT_ECUDA;
}

// On any failure the copies already queued on the plan's streams still touch the caller's host buffers and the plan's
// staging memory: drain all three streams before reporting the error.
static int exec_host_pipelined(ozfft_plan p, const char *hin, char *hout, cudaStream_t st) {
    const int rc = exec_host_pipelined_body(p, hin, hout, st);
    if (rc != OZFFT_OK) {
        const std::string keep = g_err;
        if (p->s_in) cudaStreamSynchronize(p->s_in);
        if (p->s_out) cudaStreamSynchronize(p->s_out);
        cudaStreamSynchronize(st);
        set_err(keep);
    }
    return rc;
}

int ozfft_exec_host(ozfft_plan p, const void *host_in, void *host_out, void *stream) {
    if (!valid(p)) { set_err("invalid or destroyed plan"); return OZFFT_EINVAL; }
    if (!host_in || !host_out) { set_err("null host pointer"); return OZFFT_EINVAL; }
    const size_t bytes = (size_t)p->count * 16;
    if (!p->h_in) {
        if (!cuda_ok(cudaMalloc(&p->h_in, bytes), "cudaMalloc(staging in)")) return OZFFT_ECUDA;
        if (!cuda_ok(cudaMalloc(&p->h_out, bytes), "cudaMalloc(staging out)")) { cudaFree(p->h_in); p->h_in = nullptr; return OZFFT_ECUDA; }
        p->dev_bytes += 2 * bytes;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (p->pipelined && !getenv("OZFFT_NO_PIPELINE")) return exec_host_pipelined(p, (const char *)host_in, (char *)host_out, st);
    if (!cuda_ok(cudaMemcpyAsync(p->h_in, host_in, bytes, cudaMemcpyHostToDevice, st), "H2D")) return OZFFT_ECUDA;
    int rc = run_stages(p, p->stages, 0, p->stages.size(), p->h_in, p->h_out, st);
    if (rc) return rc;
    if (!cuda_ok(cudaMemcpyAsync(host_out, p->h_out, bytes, cudaMemcpyDeviceToHost, st), "D2H")) return OZFFT_ECUDA;
    return cuda_ok(cudaStreamSynchronize(st), "cudaStreamSynchronize") ? OZFFT_OK : OZFFT_ECUDA;
}

void ozfft_plan_destroy(ozfft_plan p) {
    {
        std::lock_guard<std::mutex> lk(g_plans_mu);
        if (!p || !g_plans.erase(p)) return;  // NULL, unknown or already destroyed: no-op
    }
    for (void *d : p->dev_allocs) cudaFree(d);
    if (p->work) cudaFree(p->work);
    if (p->ring) cudaFree(p->ring);
    if (p->ctr) cudaFree(p->ctr);
    if (p->h_in) cudaFree(p->h_in);
    if (p->h_out) cudaFree(p->h_out);
    if (p->s_in) {
        cudaStreamDestroy(p->s_in);
        cudaStreamDestroy(p->s_out);
        for (int i = 0; i < PIPE; i++) { cudaEventDestroy(p->ev_in[i]); cudaEventDestroy(p->ev_out[i]); }
        cudaEventDestroy(p->ev_start);
    }
    p->magic = 0;
    delete p;
}

const char *ozfft_last_error(void) { return g_err.c_str(); }

int ozfft_probe_crt(int n, const void *d_residues, void *d_out, int variant, void *stream) {
    if (n <= 0 || !d_residues || !d_out || (variant != 0 && variant != 1)) { set_err("ozfft_probe_crt: bad argument"); return OZFFT_EINVAL; }
    DevConsts hc;
    fill_consts(hc);
    DevConsts *dc = nullptr;
    if (!cuda_ok(cudaMalloc(&dc, sizeof(hc)), "cudaMalloc(consts)")) return OZFFT_ECUDA;
    bool ok = cuda_ok(cudaMemcpy(dc, &hc, sizeof(hc), cudaMemcpyHostToDevice), "cudaMemcpy(consts)") && stage_tc_prepare(hc);
    if (ok) {
        probe_crt_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(variant, n, (const uint16_t *)d_residues, (uint32_t *)d_out, dc);
        ok = cuda_ok(cudaGetLastError(), "probe_crt_kernel launch") && cuda_ok(cudaStreamSynchronize((cudaStream_t)stream), "probe_crt_kernel");
    }
    cudaFree(dc);
    return ok ? OZFFT_OK : OZFFT_ECUDA;
}

size_t ozfft_debug_bf_tables(int K, int fusedN, int sign, void *h_B, void *h_C, void *h_PA) {
    if (K < 2 || K > 32 || (K & (K - 1)) || (sign != 1 && sign != -1) || (fusedN && fusedN != 32 * K)) return 0;
    std::vector<uint8_t> B;
    std::vector<uint32_t> Cc;
    build_mat_bf(B, Cc, K, fusedN, sign, twiddles());
    if (h_B) memcpy(h_B, B.data(), B.size());
    if (h_C) memcpy(h_C, Cc.data(), Cc.size() * 4);
    if (h_PA) {
        CrtConsts C;
        build_crt(C);
        build_pa_bf((uint8_t *)h_PA, C);
    }
    return B.size();
}

int ozfft_debug_timers(unsigned long long *h) {
#ifdef OZFFT_PIPE_TIMERS
    return cudaMemcpyFromSymbol(h, g_bf_dbg, sizeof(g_bf_dbg)) == cudaSuccess ? 160 : 0;
#else
    (void)h;
    return 0;
#endif
}

int ozfft_debug_fuse_sequence(int block, int lag, int groups, int *stage, int *group) {
    if (block < 0 || groups < 1 || lag < 1 || lag > groups || block >= 2 * groups || !stage || !group) return OZFFT_EINVAL;
    bf_sequence(block, lag, groups, *stage, *group);
    return OZFFT_OK;
}

// ---------------------------------------------------------------------------------------------------- no-allocation entry point
// ozfft_fft1d_1024_static: the batched 1-D transform of length 1024 (BASELINE.json config 3's shape) for callers that cannot
// call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it) and therefore cannot create a plan.
// It runs the fused-axis launch of the byte-fed kernel (stage_bf.cuh BfFuse) with its scratch -- the ring of Y' slots and the
// per-group counters -- in the file-scope array below instead of plan-owned memory, and with the (constant) operand tables in
// a second file-scope array filled at set-up.  Nothing here calls cudaMalloc / cudaFree or an allocating library routine.
// In host code the array names are host-side stand-ins, not device addresses: the addresses come from
// cudaGetSymbolAddress, once per device, with that device current (static_setup).
constexpr int ST_RING_SLOTS = 8, ST_LAG = 4;                      // ring of 8 slots x 2 MiB, second stage 4 groups behind the first
constexpr int ST_MAX_GROUPS = OZFFT_STATIC_MAX_BATCH / 128;       // 512 groups of 128 pencils
constexpr size_t ST_CTR_BYTES = (size_t)2 * ST_MAX_GROUPS * 4;    // store / read counters, one pair per group
constexpr size_t ST_SCRATCH_BYTES = ST_CTR_BYTES + (size_t)ST_RING_SLOTS * BF_GROUP_ELEMS * 16;
static_assert(ST_SCRATCH_BYTES == OZFFT_STATIC_SCRATCH_BYTES, "ozfft.h states the size of the static scratch");
static __device__ __align__(256) unsigned char g_static_scratch[ST_SCRATCH_BYTES];
// operand tables per direction: [F_32 planes | 32 fused planes | offset constants 1 | offset constants 2], then the Phase-A matrix
constexpr size_t ST_MAT1 = bf_mat_bytes(32), ST_MAT2 = 32 * bf_mat_bytes(32), ST_C1 = 32 * 16, ST_C2 = 32 * 32 * 16;
constexpr size_t ST_SIGN_BYTES = ST_MAT1 + ST_MAT2 + ST_C1 + ST_C2;
static __device__ __align__(256) unsigned char g_static_tables[2 * ST_SIGN_BYTES + BF_PA_BYTES];

namespace {
struct StaticDev { bool ready = false; int sms = 0; unsigned char *scratch = nullptr, *tables = nullptr; };
std::mutex g_static_mu;
std::map<int, StaticDev> g_static_dev;

// once per device, with that device current: symbol addresses, kernel attributes, constant bank, tables for both directions
int static_setup(StaticDev *&out) {
    int dev = 0;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return OZFFT_ECUDA;
    std::lock_guard<std::mutex> lk(g_static_mu);
    StaticDev &d = g_static_dev[dev];
    out = &d;
    if (d.ready) return OZFFT_OK;
    int major = 0;
    if (!cuda_ok(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev), "cudaDeviceGetAttribute") ||
        !cuda_ok(cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute")) return OZFFT_ECUDA;
    if (major != 10) { set_err("ozfft needs an sm_100 device (B200); no fallback path exists"); return OZFFT_ECUDA; }
    if (!cuda_ok(cudaGetSymbolAddress((void **)&d.scratch, g_static_scratch), "cudaGetSymbolAddress(scratch)") ||
        !cuda_ok(cudaGetSymbolAddress((void **)&d.tables, g_static_tables), "cudaGetSymbolAddress(tables)")) return OZFFT_ECUDA;
    DevConsts hc;
    fill_consts(hc);
    if (!stage_tc_prepare(hc) || !stage_bf_prepare()) { set_err("kernel attribute setup failed"); return OZFFT_ECUDA; }
    for (int si = 0; si < 2; si++) {  // si = 0: sign -1 (forward), 1: sign +1
        unsigned char *base = d.tables + (size_t)si * ST_SIGN_BYTES;
        std::vector<uint8_t> B;
        std::vector<uint32_t> C;
        build_mat_bf(B, C, 32, 0, si ? 1 : -1, twiddles());
        if (B.size() != ST_MAT1 || C.size() * 4 != ST_C1) { set_err("static tables: unexpected table size"); return OZFFT_ECUDA; }
        if (!cuda_ok(cudaMemcpy(base, B.data(), ST_MAT1, cudaMemcpyHostToDevice), "cudaMemcpy(static tables)") ||
            !cuda_ok(cudaMemcpy(base + ST_MAT1 + ST_MAT2, C.data(), ST_C1, cudaMemcpyHostToDevice), "cudaMemcpy(static tables)")) return OZFFT_ECUDA;
        build_mat_bf(B, C, 32, 1024, si ? 1 : -1, twiddles());
        if (B.size() != ST_MAT2 || C.size() * 4 != ST_C2) { set_err("static tables: unexpected table size"); return OZFFT_ECUDA; }
        if (!cuda_ok(cudaMemcpy(base + ST_MAT1, B.data(), ST_MAT2, cudaMemcpyHostToDevice), "cudaMemcpy(static tables)") ||
            !cuda_ok(cudaMemcpy(base + ST_MAT1 + ST_MAT2 + ST_C1, C.data(), ST_C2, cudaMemcpyHostToDevice), "cudaMemcpy(static tables)")) return OZFFT_ECUDA;
    }
    CrtConsts Cc;
    build_crt(Cc);
    std::vector<uint8_t> pa(BF_PA_BYTES);
    build_pa_bf(pa.data(), Cc);
    if (!cuda_ok(cudaMemcpy(d.tables + 2 * ST_SIGN_BYTES, pa.data(), BF_PA_BYTES, cudaMemcpyHostToDevice), "cudaMemcpy(static tables)")) return OZFFT_ECUDA;
    d.ready = true;
    return OZFFT_OK;
}
}  // namespace

int ozfft_static_setup(void) {
    StaticDev *d = nullptr;
    return static_setup(d);
}

int ozfft_fft1d_1024_static(int batch, int sign, const void *in, void *out, void *stream) {
    if (sign != -1 && sign != 1) { set_err("sign must be -1 (forward) or +1 (inverse)"); return OZFFT_EINVAL; }
    if (batch < 128 || batch % 128 || batch > OZFFT_STATIC_MAX_BATCH) {
        set_err("ozfft_fft1d_1024_static: batch must be a multiple of 128 in [128, " + std::to_string(OZFFT_STATIC_MAX_BATCH) +
                "] (the static scratch holds counters for " + std::to_string(ST_MAX_GROUPS) + " groups of 128 pencils); use a plan for other sizes");
        return OZFFT_EINVAL;
    }
    if (!check_ptrs(in, out)) return OZFFT_EINVAL;
    StaticDev *d = nullptr;
    int rc = static_setup(d);  // a no-op after the first call on this device
    if (rc) return rc;
    // geometry: the plan code's own (add_axis), fed with the static tables so that it finds them and uploads nothing
    const int si = sign == 1 ? 1 : 0;
    unsigned char *base = d->tables + (size_t)si * ST_SIGN_BYTES;
    MatMap mats;
    MatSet m1{}, m2{};
    m1.bf = base; m1.ctab = base + ST_MAT1 + ST_MAT2;
    m2.bf = base + ST_MAT1; m2.ctab = base + ST_MAT1 + ST_MAT2 + ST_C1;
    mats[MatKey{32, 0}] = m1;
    mats[MatKey{32, 1024}] = m2;
    ozfft_plan_s tmp{};
    tmp.variant = 2; tmp.sign = sign; tmp.max_groups = 0;
    std::vector<StageLaunch> st;
    if (!add_axis(&tmp, AxisDesc{true, batch, 1024, 1}, 0, mats, st, false, 0, true) || st.size() != 1 || !st[0].fused) {
        set_err("ozfft_fft1d_1024_static: internal geometry error");
        return OZFFT_EINVAL;
    }
    BfFuse f = st[0].fuse;
    f.wr_done = (unsigned int *)d->scratch;
    f.rd_done = f.wr_done + ST_MAX_GROUPS;
    f.ring = (uint4 *)(d->scratch + ST_CTR_BYTES);
    f.Lg = ST_LAG < f.G ? ST_LAG : f.G;
    f.R = ST_RING_SLOTS;
    // stage_bf_launch_fused zeroes the group counters on the stream (memset, no allocation), then launches the kernel; the ring
    // needs no clearing: every slot is written before it is read
    if (!stage_bf_launch_fused(st[0].g, f, in, out, st[0].mat_bf, st[0].ctab_bf, d->tables + 2 * ST_SIGN_BYTES, d->sms, (cudaStream_t)stream)) {
        set_err(std::string("stage_bf_kernel (static scratch) launch: ") + cudaGetErrorString(cudaGetLastError()));
        return OZFFT_ECUDA;
    }
    return OZFFT_OK;
}

uint64_t ozfft_twiddle_checksum(void) { return twiddle_fnv(twiddles()); }

int ozfft_plan_num_launches(ozfft_plan p) { return valid(p) ? (int)p->stages.size() : -1; }

size_t ozfft_plan_device_bytes(ozfft_plan p) { return valid(p) ? p->dev_bytes : 0; }

}  // extern "C"
