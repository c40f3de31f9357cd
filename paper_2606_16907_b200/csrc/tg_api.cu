// libtangram host side: C-ABI entry points (include/tangram.h), instance ownership, workspace
// carving and kernel launches.  No CPU fallback: every compute path ends in a CUDA launch.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <mutex>
#include <string>
#include <algorithm>
#include <vector>

#include "tg_common.cuh"
#include "tg_prep.cuh"
// the persistent solver, twice: core path only / with the variants of SURVEY.md §8(f) (see the head of tg_solve.cuh)
#define TG_SOLVE_NS tgcore
#define TG_VAR 0
#include "tg_solve.cuh"
#undef TG_SOLVE_NS
#undef TG_VAR
#define TG_SOLVE_NS tgfull
#define TG_VAR 1
#include "tg_solve.cuh"
#undef TG_SOLVE_NS
#undef TG_VAR
#include "tg_islands.cuh"

// One device allocation shared by the instances of a tg_instance_create_batch call; freed with the last of them.
struct TgBatchBlock {
    char* base = nullptr;
    std::atomic<int> refs{0};
};

struct tg_instance {
    TgBatchBlock* block = nullptr;                   // nullptr: the instance owns its allocation (time_us is its base)
    int32_t L, K, P, m, act_mb, NS;
    int device;
    int32_t *time_us, *mem_mb, *gpus, *cap_mb, *bw;  // device
    int32_t* actmem;                                 // device, or nullptr (tg_instance_set_actmem)
    int32_t* cls = nullptr;                          // device block [classOf NS | class time NC*K*P | class mem NC*K*P], or nullptr
    int32_t nClasses = 0;                            //   (tg_instance_create_classes; dropped when the instance is pruned or gets
    bool toeplitz = false;                           //   footprint / stage tables: they work on the expanded tables)
    int32_t nAct = 0;                                // tg_instance_set_boundary_act: distinct activation sizes (0 = scalar act_mb)
    int32_t actVal[TG_MAX_ACT] = {0, 0, 0, 0, 0, 0, 0, 0};
    uint8_t clsOf[256] = {0};                        // size class of boundary b
    int32_t* slow = nullptr;                         // device, or nullptr (tg_instance_set_stages): slowest internal stage [NS][K][P]
    int32_t* qst = nullptr;                          // device, behind slow: internal stage counts [NS][K][P]
    int32_t xbound;                                  // tg_instance_set_transfer_bound
};

namespace {

thread_local std::string g_err;

tg_status fail(tg_status st, const std::string& msg) {
    g_err = msg;
    return st;
}

#define TG_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? TG_ERR_OOM : TG_ERR_CUDA,                \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                       \
    } while (0)

struct DeviceState {
    bool ready = false;
    int numSMs = 0;
    int smemOptin = 0;
    int smemPerSM = 0;
    int ctasPerSM = 0;    // co-resident CTAs of the solver per SM
    int dynSmem = 0;      // dynamic shared memory of one solver CTA
    uint64_t budget = 0;  // bytes the DP scratch may take (from cudaMemGetInfo; refreshed every 64 solves or after a failed allocation)
    int budgetAge = 0;
    uint16_t* rankOf = nullptr;
    uint16_t* maskOf = nullptr;
    cudaMemPool_t pool = nullptr;   // the library's own stream-ordered pool for per-call workspaces
    cudaStream_t up[4] = {nullptr, nullptr, nullptr, nullptr};   // upload streams of tg_instance_create_batch
    cudaEvent_t upEv[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
};
std::mutex g_mu;
int g_gallopMax = [] { const char* e = getenv("TG_GALLOP_MAX"); int v = e ? atoi(e) : 10; return v < 1 ? 1 : (v > 16 ? 16 : v); }();
// DPs per instance and scheduler round (speculation width of the threshold search / sweep)
int g_wishFloor = [] { const char* e = getenv("TG_WISH_FLOOR"); int v = e ? atoi(e) : 8; return v < 1 ? 1 : (v > 12 ? 12 : v); }();
int g_wishCap = [] { const char* e = getenv("TG_WISH_CAP"); int v = e ? atoi(e) : 12; return v < 8 ? 8 : (v > TG_MAX_WISH ? TG_MAX_WISH : v); }();
int g_queueWish = [] { const char* e = getenv("TG_QUEUE_WISH"); int v = e ? atoi(e) : 6; return v < 1 ? 1 : (v > 12 ? 12 : v); }();
int g_wishMax = [] { const char* e = getenv("TG_WISH_MAX"); int v = e ? atoi(e) : 64; return v < 1 ? 1 : (v > TG_MAX_WISH ? TG_MAX_WISH : v); }();
DeviceState g_dev[64];

tg_status deviceInit(int dev, DeviceState** out) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (dev < 0 || dev >= 64) return fail(TG_ERR_CUDA, "device ordinal out of range");
    DeviceState& D = g_dev[dev];
    if (!D.ready) {
        cudaDeviceProp prop;
        TG_CUDA(cudaGetDeviceProperties(&prop, dev));
        D.numSMs = prop.multiProcessorCount;
        D.smemOptin = int(prop.sharedMemPerBlockOptin);
        D.smemPerSM = int(prop.sharedMemPerMultiprocessor);
        int coop = 0;
        TG_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        if (!coop) return fail(TG_ERR_CUDA, "device lacks cooperative launch");
        // rankOf[mask] = colexicographic rank inside its popcount class (masks of one popcount ordered by value)
        std::vector<uint16_t> rankOf(65536);
        uint16_t binom[17][17];
        memset(binom, 0, sizeof(binom));
        for (int n = 0; n <= 16; ++n) {
            binom[n][0] = 1;
            for (int r = 1; r <= n; ++r) binom[n][r] = uint16_t(binom[n - 1][r - 1] + (r <= n - 1 ? binom[n - 1][r] : 0));
        }
        uint32_t fill[17], popOff[18];
        memset(fill, 0, sizeof(fill));
        popOff[0] = 0;
        for (int r = 0; r <= 16; ++r) popOff[r + 1] = popOff[r] + binom[16][r];
        std::vector<uint16_t> maskOf(65536);   // masks ordered by (popcount, value): the inverse of rankOf
        for (uint32_t mk = 0; mk < 65536; ++mk) {
            const int r = __builtin_popcount(mk);
            rankOf[mk] = uint16_t(fill[r]);
            maskOf[popOff[r] + fill[r]] = uint16_t(mk);
            ++fill[r];
        }
        TG_CUDA(cudaMalloc(&D.rankOf, 2 * 65536 * sizeof(uint16_t)));
        D.maskOf = D.rankOf + 65536;
        TG_CUDA(cudaMemcpy(D.rankOf, rankOf.data(), 65536 * sizeof(uint16_t), cudaMemcpyHostToDevice));
        TG_CUDA(cudaMemcpy(D.maskOf, maskOf.data(), 65536 * sizeof(uint16_t), cudaMemcpyHostToDevice));
        TG_CUDA(cudaMemcpyToSymbol(tgPopOff, popOff, sizeof(popOff)));
        TG_CUDA(cudaMemcpyToSymbol(tgBinom, binom, sizeof(binom)));
        TG_CUDA(cudaFuncSetAttribute(tgPrepareKernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TG_SORT_SMEM_MAX * 4));
        cudaFuncAttributes fa, fb;
        TG_CUDA(cudaFuncGetAttributes(&fa, tgcore::tgSolveKernel));
        TG_CUDA(cudaFuncGetAttributes(&fb, tgfull::tgSolveKernel));
        // TG_CTAS_PER_SM co-resident CTAs share the SM's shared memory (each CTA also pays 1 KB of system reserve)
        int dyn = std::min(D.smemOptin, D.smemPerSM / TG_CTAS_PER_SM) - int(std::max(fa.sharedSizeBytes, fb.sharedSizeBytes)) - 1024;
        dyn &= ~1023;
        if (dyn < 48 * 1024) return fail(TG_ERR_CUDA, "not enough shared memory per block for the solver");
        TG_CUDA(cudaFuncSetAttribute(tgcore::tgSolveKernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn));
        TG_CUDA(cudaFuncSetAttribute(tgfull::tgSolveKernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn));
        int occ = 0, occ2 = 0;
        TG_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, tgcore::tgSolveKernel, TG_NT, size_t(dyn)));
        TG_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, tgfull::tgSolveKernel, TG_NT, size_t(dyn)));
        if (std::min(occ, occ2) < TG_CTAS_PER_SM) return fail(TG_ERR_CUDA, "solver kernel: fewer co-resident CTAs per SM than it was built for");
        D.ctasPerSM = TG_CTAS_PER_SM;
        D.dynSmem = dyn;
        // Per-call workspaces come from a pool of the library's own (the device's default pool, which the embedding
        // framework may share, is left as it is).  Freed workspaces stay cached up to the release threshold, so
        // back-to-back solves do not go to the driver; anything above it returns to the device at the next synchronisation.
        {
            cudaMemPoolProps props;
            memset(&props, 0, sizeof(props));
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = dev;
            TG_CUDA(cudaMemPoolCreate(&D.pool, &props));
            // (the largest workspace is the DP scratch, capped at 12 GB in prepare(): a lower threshold would hand it back
            // to the driver at every synchronisation and map it again on the next call -- measured 125 ms a call)
            uint64_t thr = 14ull << 30;
            if (const char* e = getenv("TG_POOL_KEEP_MB")) thr = uint64_t(std::max(0ll, atoll(e))) << 20;
            TG_CUDA(cudaMemPoolSetAttribute(D.pool, cudaMemPoolAttrReleaseThreshold, &thr));
        }
        for (int q = 0; q < 4; ++q) TG_CUDA(cudaStreamCreateWithFlags(&D.up[q], cudaStreamNonBlocking));
        for (int q = 0; q < 5; ++q) TG_CUDA(cudaEventCreateWithFlags(&D.upEv[q], cudaEventDisableTiming));
        D.ready = true;
    }
    *out = &D;
    return TG_OK;
}

inline size_t alignUp(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Stream-ordered device memory from the library's own pool (instance tables as well as per-call workspaces: memory freed
// into the device's DEFAULT pool goes back to the driver at the next synchronisation and is mapped again on the next
// allocation -- an end-to-end loop that creates and destroys 385 MB of tables per step then stalls for up to a second now
// and then).
cudaError_t poolAlloc(void** p, size_t bytes, cudaStream_t st) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    DeviceState* D = nullptr;
    if (deviceInit(dev, &D) != TG_OK) return cudaErrorInitializationError;
    return cudaMallocFromPoolAsync(p, bytes, D->pool, st);
}

struct Carver {
    size_t off = 0;
    size_t take(size_t bytes, size_t align = 256) {
        off = alignUp(off, align);
        const size_t o = off;
        off += bytes;
        return o;
    }
};

bool isDevicePtr(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

struct Workspace {
    char* base = nullptr;           // freed (stream-ordered) when the workspace goes out of scope, on every path
    cudaStream_t stream = nullptr;
    ~Workspace() { if (base) cudaFreeAsync(base, stream); }
    size_t bytes = 0;
    TgInstDev* inst = nullptr;
    TgSolveCtx ctx;
    tg_result* outDev = nullptr;
    int dynSmem = 0;
    int numCtas = 0;
    bool variants = false;          // an instance of the batch uses a SURVEY 8(f) variant: launch the full kernel
};

// Lays out the per-call workspace, uploads the instance records and runs loader + prepare.
thread_local cudaEvent_t g_evL0 = nullptr, g_evL1 = nullptr;  // bracket the last loader kernel of this thread

tg_status prepare(tg_instance* const* instances, int n, bool needSolve, cudaStream_t st, Workspace& W) {
    if (!instances) return fail(TG_ERR_NULL, "instances is NULL");
    if (n < 1 || n > 65535) return fail(TG_ERR_SHAPE, "n must be in [1, 65535]");
    for (int i = 0; i < n; ++i)
        if (!instances[i]) return fail(TG_ERR_NULL, "instances[" + std::to_string(i) + "] is NULL");
    int dev = 0;
    TG_CUDA(cudaGetDevice(&dev));
    for (int i = 0; i < n; ++i)
        if (instances[i]->device != dev) return fail(TG_ERR_CUDA, "instance was created on another device");
    DeviceState* D;
    tg_status s = deviceInit(dev, &D);
    if (s != TG_OK) return s;

    Carver cv;
    const size_t oInst = cv.take(sizeof(TgInstDev) * n);
    std::vector<TgInstDev> h(n);
    std::vector<size_t> oCdT(n), oXa(n), oCd(n), oThr(n), oArgp(n), oCand(n), oSort(n), oSort2(n), oSuf(n), oSufA(n), oEI(n), oEF(n);
    int maxCells = 0, maxLp = 4, maxK = 1;
    uint64_t maxFull = 0;
    size_t denseCs = 0;
    for (int i = 0; i < n; ++i) {
        const tg_instance& t = *instances[i];
        TgInstDev& I = h[i];
        memset(&I, 0, sizeof(I));
        I.time_us = t.time_us; I.mem_mb = t.mem_mb; I.cap_mb = t.cap_mb; I.bw_gbps = t.bw;
        I.actmem_mb = t.actmem;
        I.nDepth = t.actmem ? t.K : 1;
        if (t.actmem || t.slow || t.nAct) W.variants = true;
        if (t.cls) {
            const size_t nC4 = size_t(t.nClasses) * t.K * t.P * 4;
            I.classOf = t.cls;
            I.ctime = reinterpret_cast<const int32_t*>(reinterpret_cast<const char*>(t.cls) + alignUp(size_t(t.NS) * 4, 256));
            I.cmem = reinterpret_cast<const int32_t*>(reinterpret_cast<const char*>(I.ctime) + alignUp(nC4, 256));
            I.toeplitz = t.toeplitz ? 1 : 0;
        }
        I.slow_us = t.slow;
        I.nLayers = t.slow ? t.P : 0;
        I.nTables = std::max(std::max(I.nDepth, I.nLayers), 1);
        I.xbound = t.xbound;
        I.nAct = t.nAct;
        memcpy(I.actVal, t.actVal, sizeof(I.actVal));
        memcpy(I.clsOf, t.clsOf, sizeof(I.clsOf));
        I.L = t.L; I.K = t.K; I.P = t.P; I.m = t.m; I.act_mb = t.act_mb; I.NS = t.NS;
        I.Lp = (t.L + 3) & ~3;
        I.triG = int(tgGOff(t.L, t.L + 1));
        const int cells = t.NS * t.K;
        int cap = 2;
        while (cap < cells) cap <<= 1;
        I.sortCap = cap;
        for (int k = 0; k < TG_MAX_K; ++k) I.cminAll[k] = TG_INFU;
        I.maxKey = 0;
        I.phase = TG_PH_NEW;
        I.incIdx = -1; I.hiFeas = -1; I.loInf = -1; I.specIdx = -1; I.specItem = -1;
        uint64_t mx = 1;
        {   // widest wavefront and full table in rows
            uint64_t binom[17][17];
            memset(binom, 0, sizeof(binom));
            for (int a = 0; a <= 16; ++a) { binom[a][0] = 1; for (int r = 1; r <= a; ++r) binom[a][r] = binom[a - 1][r - 1] + binom[a - 1][r]; }
            for (int r = 0; r < t.K; ++r) mx = std::max<uint64_t>(mx, binom[t.K][r] * uint64_t(t.K - r));
        }
        const uint64_t full = uint64_t(t.K) * (1ull << (t.K - 1)) * uint64_t(I.Lp);
        I.fullWords = full;
        maxFull = std::max<uint64_t>(maxFull, std::max<uint64_t>(full, 2 * mx * uint64_t(I.Lp)));
        denseCs = std::max<size_t>(denseCs, size_t(t.K) * tgSOff(t.L, t.L));
        maxCells = std::max(maxCells, cells);
        maxLp = std::max(maxLp, int(I.Lp));
        maxK = std::max(maxK, int(t.K));
        const size_t nd = size_t(I.nTables);
        oCd[i] = cv.take(nd * size_t(t.K) * I.triG * 4);
        oThr[i] = I.nLayers ? cv.take(nd * size_t(t.K) * I.triG * 4) : 0;
        oArgp[i] = cv.take(nd * size_t(cells));
        oCdT[i] = (t.cls && t.toeplitz) ? cv.take(size_t(t.K) * (t.L + 2) * 4) : 0;
        oXa[i] = t.nAct ? cv.take(size_t(t.nAct) * TG_MAX_K * TG_MAX_K * 4) : 0;
        const size_t nKeys = nd * size_t(cells) + size_t(t.K) * t.K * std::max(t.nAct, 1);   // every reduced cost + (transfer bound) every transfer time
        oCand[i] = cv.take(nKeys * 4);
        oSort[i] = cv.take(nKeys * 4);
        oSort2[i] = cv.take(nKeys * 4);
        oSuf[i] = cv.take(size_t(t.K) * (t.L + 2) * 4);
        oSufA[i] = cv.take(size_t(t.K) * (t.L + 2) * 4);
        oEI[i] = cv.take(size_t(TG_MAX_EVAL) * 4);
        oEF[i] = cv.take(size_t(TG_MAX_EVAL) * 4);
    }
    const size_t oItems = cv.take(sizeof(TgItem) * TG_QCAP);
    const size_t oKeys = cv.take(sizeof(unsigned long long) * TG_QCAP);
    const size_t oCtrl = cv.take(sizeof(TgCtrl));
    const size_t oOut = cv.take(sizeof(tg_result) * n);
    const size_t oSpec = cv.take(sizeof(tg_result) * TG_QCAP);
    const size_t oSeq = cv.take(sizeof(uint32_t) * TG_QCAP);
    // DP scratch: nSlots slots, each able to hold every level of the largest instance.  A slot
    // belongs to one team (team mode) or one CTA (solo mode) for the duration of a DP.
    const int numCtas = D->numSMs * D->ctasPerSM;
    const uint64_t slotWords = alignUp(size_t(maxFull) + 1024, 1024);
    int nSlots = 0;
    if (needSolve) {
        uint64_t budget;
        {
            std::lock_guard<std::mutex> lk(g_mu);   // (solves may come from several host threads)
            if (D->budget == 0 || ++D->budgetAge >= 64) {   // (the query costs tens of microseconds: not on every solve)
                size_t freeB = 0, totalB = 0;
                TG_CUDA(cudaMemGetInfo(&freeB, &totalB));
                D->budget = std::min<uint64_t>(uint64_t(freeB) * 6 / 10, 12ull << 30);   // bytes
                D->budgetAge = 0;
            }
            budget = D->budget;
        }
        nSlots = int(std::min<uint64_t>(uint64_t(numCtas), budget / (slotWords * 4)));
        if (nSlots < 1) nSlots = 1;   // let the allocation decide
    }
    const size_t oBar = cv.take(sizeof(uint32_t) * size_t(std::max(nSlots, 1)));
    const size_t oScratch = cv.take(size_t(slotWords) * 4 * size_t(nSlots), 4096);
    W.bytes = cv.off + 4096;
    {
        W.stream = st;
        const cudaError_t ea = cudaMallocFromPoolAsync(reinterpret_cast<void**>(&W.base), W.bytes, D->pool, st);
        if (ea != cudaSuccess) {
            { std::lock_guard<std::mutex> lk(g_mu); D->budget = 0; }   // measure again on the next call
            cudaGetLastError();
            return fail(ea == cudaErrorMemoryAllocation ? TG_ERR_OOM : TG_ERR_CUDA, std::string("workspace allocation: ") + cudaGetErrorString(ea));
        }
    }
    for (int i = 0; i < n; ++i) {
        h[i].cd = reinterpret_cast<uint32_t*>(W.base + oCd[i]);
        h[i].thr = h[i].nLayers ? reinterpret_cast<uint32_t*>(W.base + oThr[i]) : nullptr;
        h[i].cdT = (h[i].classOf && h[i].toeplitz) ? reinterpret_cast<uint32_t*>(W.base + oCdT[i]) : nullptr;
        h[i].xAct = h[i].nAct ? reinterpret_cast<uint32_t*>(W.base + oXa[i]) : nullptr;
        h[i].argp = reinterpret_cast<uint8_t*>(W.base + oArgp[i]);
        h[i].cand = reinterpret_cast<uint32_t*>(W.base + oCand[i]);
        h[i].sortbuf = reinterpret_cast<uint32_t*>(W.base + oSort[i]);
        h[i].sortbuf2 = reinterpret_cast<uint32_t*>(W.base + oSort2[i]);
        h[i].sufMin = reinterpret_cast<uint32_t*>(W.base + oSuf[i]);
        h[i].sufMinAll = reinterpret_cast<uint32_t*>(W.base + oSufA[i]);
        h[i].eIdx = reinterpret_cast<int32_t*>(W.base + oEI[i]);
        h[i].eF = reinterpret_cast<uint32_t*>(W.base + oEF[i]);
    }
    W.inst = reinterpret_cast<TgInstDev*>(W.base + oInst);
    W.outDev = reinterpret_cast<tg_result*>(W.base + oOut);
    W.numCtas = numCtas;
    TG_CUDA(cudaMemcpyAsync(W.inst, h.data(), sizeof(TgInstDev) * n, cudaMemcpyHostToDevice, st));
    TG_CUDA(cudaMemsetAsync(W.base + oCtrl, 0, sizeof(TgCtrl), st));
    if (n >= TG_WIDE_MIN_INST && n <= TG_QUEUE_MAX_INST)   // the publication flags of queue mode (the only mode that reads them)
        TG_CUDA(cudaMemsetAsync(W.base + oSeq, 0, sizeof(uint32_t) * TG_QCAP, st));

    // shared-memory split of the solver: warp-private row buffers (H rows + two source buffers =
    // 2*Kmax rows of Lp+8 words per warp) vs staged cost tables (at least a quarter of the total)
    W.dynSmem = D->dynSmem;
    const int totalWords = W.dynSmem / 4;
    TgSolveCtx& c = W.ctx;
    memset(&c, 0, sizeof(c));
    c.dynWords = totalWords & ~3;
    c.inst = W.inst; c.nInst = n;
    c.items = reinterpret_cast<TgItem*>(W.base + oItems);
    c.keys = reinterpret_cast<unsigned long long*>(W.base + oKeys);
    c.scratch = reinterpret_cast<uint32_t*>(W.base + oScratch);
    c.slotWords = slotWords; c.nSlots = nSlots;
    c.slotBar = reinterpret_cast<uint32_t*>(W.base + oBar);
    c.wishMax = g_wishMax;
    c.queueWish = g_queueWish;
    c.gallopMax = g_gallopMax;
    c.wishCap = g_wishCap;
    c.wishFloor = g_wishFloor;
    c.ctrl = reinterpret_cast<TgCtrl*>(W.base + oCtrl);
    c.rankOf = D->rankOf;
    c.maskOf = D->maskOf;
    c.specOut = reinterpret_cast<tg_result*>(W.base + oSpec);
    c.itemSeq = reinterpret_cast<uint32_t*>(W.base + oSeq);

    // loader grid: 256 * U cells per CTA, U = TG_LOAD_U when that still gives every SM two CTAs, else 1; the
    // batched-load path is compiled for P = 4 and P = 8 (picked from the first instance; instances of another
    // shape take the kernel's cell-at-a-time path)
    const int ctasU = (maxCells + 256 * TG_LOAD_U - 1) / (256 * TG_LOAD_U);
    const bool wide = int64_t(ctasU) * n >= 2 * D->numSMs;
    const dim3 g(wide ? ctasU : (maxCells + 255) / 256, n);
    const int P0 = instances[0]->P;
    if (!g_evL0) { TG_CUDA(cudaEventCreate(&g_evL0)); TG_CUDA(cudaEventCreate(&g_evL1)); }
    TG_CUDA(cudaEventRecord(g_evL0, st));
    // a batch of plain instances with P = 4 or 8 that fills the GPU takes the row-group loader (reduced costs transposed
    // through shared memory, 32-byte runs into the diagonal-major tables)
    bool rows = wide && (P0 == 4 || P0 == 8) && size_t(maxK) * (maxLp) * TG_LOAD_RG * 4 <= size_t(96) * 1024;
    for (int i = 0; i < n && rows; ++i) rows = instances[i]->P == P0 && !instances[i]->actmem && !instances[i]->slow;
    if (rows) {
        int maxL = 1;
        for (int i = 0; i < n; ++i) maxL = std::max(maxL, int(instances[i]->L));
        const dim3 gr((maxL + TG_LOAD_RG - 1) / TG_LOAD_RG, n);
        const size_t sh = size_t(maxK) * maxL * TG_LOAD_RG * 4;
        if (P0 == 4) {
            TG_CUDA(cudaFuncSetAttribute(tgLoadRowsKernel<1, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
            tgLoadRowsKernel<1, 4><<<gr, TG_LR_NT, sh, st>>>(W.inst);
        } else {
            TG_CUDA(cudaFuncSetAttribute(tgLoadRowsKernel<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
            tgLoadRowsKernel<2, 2><<<gr, TG_LR_NT, sh, st>>>(W.inst);
        }
    } else if (wide) {
        if (P0 == 4) tgLoadKernel<1, TG_LOAD_U><<<g, 256, 0, st>>>(W.inst);
        else if (P0 == 8) tgLoadKernel<2, TG_LOAD_U><<<g, 256, 0, st>>>(W.inst);
        else tgLoadKernel<0, TG_LOAD_U><<<g, 256, 0, st>>>(W.inst);
    } else {
        if (P0 == 4) tgLoadKernel<1, 1><<<g, 256, 0, st>>>(W.inst);
        else if (P0 == 8) tgLoadKernel<2, 1><<<g, 256, 0, st>>>(W.inst);
        else tgLoadKernel<0, 1><<<g, 256, 0, st>>>(W.inst);
    }
    TG_CUDA(cudaEventRecord(g_evL1, st));
    tgPrepareKernel<<<n, TG_PREP_NT, TG_SORT_SMEM_MAX * 4, st>>>(W.inst);
    TG_CUDA(cudaGetLastError());
    return TG_OK;
}

thread_local cudaEvent_t g_evA = nullptr, g_evB = nullptr;  // bracket the last solver kernel of this thread

tg_status launchSolve(Workspace& W, cudaStream_t st) {
    TgSolveCtx ctx = W.ctx;
    void* args[] = {&ctx};
    if (!g_evA) { TG_CUDA(cudaEventCreate(&g_evA)); TG_CUDA(cudaEventCreate(&g_evB)); }
    TG_CUDA(cudaEventRecord(g_evA, st));
    const void* kernel = W.variants ? (const void*)tgfull::tgSolveKernel : (const void*)tgcore::tgSolveKernel;
    TG_CUDA(cudaLaunchCooperativeKernel(kernel, dim3(W.numCtas), dim3(TG_NT), args, size_t(W.dynSmem), st));
    TG_CUDA(cudaEventRecord(g_evB, st));
    return TG_OK;
}

tg_status finish(Workspace& W, int n, tg_result* out, tg_solve_stats* stats, cudaStream_t st) {
    const bool outDev = isDevicePtr(out);
    bool sync = !outDev;
    tgcore::tgPoisonOnErrorKernel<<<std::max(1, std::min((n + 255) / 256, 64)), 256, 0, st>>>(W.ctx.ctrl, W.outDev, n);
    TG_CUDA(cudaMemcpyAsync(out, W.outDev, sizeof(tg_result) * n, cudaMemcpyDefault, st));
    if (stats) {
        if (!isDevicePtr(stats)) sync = true;
        TG_CUDA(cudaMemcpyAsync(&W.ctx.ctrl->stats.error_flag, &W.ctx.ctrl->errFlag, sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        TG_CUDA(cudaMemcpyAsync(stats, &W.ctx.ctrl->stats, sizeof(tg_solve_stats), cudaMemcpyDefault, st));
    }
    static const bool dbg = getenv("TG_DEBUG") != nullptr;
    if (dbg) {
        static TgCtrl hc;
        TG_CUDA(cudaMemcpyAsync(&hc, W.ctx.ctrl, sizeof(TgCtrl), cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        const int nr = int(std::min<uint64_t>(hc.stats.n_rounds, 256));
        fprintf(stderr, "[tg] rounds=%d dps=%llu\n", nr, (unsigned long long)hc.stats.n_dp);
        {
            static TgInstDev hi;
            TG_CUDA(cudaMemcpy(&hi, W.inst, sizeof(TgInstDev), cudaMemcpyDeviceToHost));
            std::vector<int32_t> e(hi.nEval > 0 ? hi.nEval : 1);
            TG_CUDA(cudaMemcpy(e.data(), hi.eIdx, sizeof(int32_t) * e.size(), cudaMemcpyDeviceToHost));
            fprintf(stderr, "[tg] inst0 prepare cycles: minima %lld sort %lld unique %lld lbIdx %lld\n", hi.prepCyc[1] - hi.prepCyc[0],
                    hi.prepCyc[2] - hi.prepCyc[1], hi.prepCyc[3] - hi.prepCyc[2], hi.prepCyc[4] - hi.prepCyc[3]);
            fprintf(stderr, "[tg] inst0: ncand=%d lbIdx=%d lowestFeasible=%d incIdx=%d nEval=%d evaluated:", hi.ncand, hi.lbIdx,
                    hi.nEval > 0 ? (e[0] & ~TG_EDONE) : -1, hi.incIdx, hi.nEval);
            for (int q = 0; q < hi.nEval && q < 48; ++q) fprintf(stderr, " %d", e[q] & ~TG_EDONE);
            fprintf(stderr, "\n");
        }
        for (int r = 0; r < nr; ++r)
            fprintf(stderr, "[tg]  round %3d items %5d  %8.1f us\n", r, hc.roundItems[r],
                    r + 1 < nr ? double(hc.roundNs[r + 1] - hc.roundNs[r]) * 1e-3 : 0.0);
        for (int r = 0; r < nr && r < 8; ++r)
            fprintf(stderr, "[tg]  round %3d scheduler cycles: fold %lld plan %lld teams %lld\n", r, hc.schedCyc[r][1] - hc.schedCyc[r][0],
                    hc.schedCyc[r][2] - hc.schedCyc[r][1], hc.schedCyc[r][3] - hc.schedCyc[r][2]);
        for (int r = 0; r < nr && r < 8; ++r)
            fprintf(stderr, "[tg]  round %3d fold/plan detail: stage-prev %lld copy-in %lld fold %lld plan %lld copy-out %lld\n", r,
                    hc.dbgCyc[r][0] - hc.schedCyc[r][0], hc.dbgCyc[r][1] - hc.dbgCyc[r][0], hc.dbgCyc[r][2] - hc.dbgCyc[r][1],
                    hc.dbgCyc[r][3] - hc.dbgCyc[r][2], hc.schedCyc[r][1] - hc.dbgCyc[r][3]);
        for (int r = 0; r < nr && r < 8; ++r) {
            if (hc.roundItems[r] > 16 || hc.roundItems[r] >= W.ctx.nSlots) continue;
            fprintf(stderr, "[tg]  round %3d items (candidate: us)", r);
            for (int t = 0; t < hc.roundItems[r]; ++t)
                fprintf(stderr, " %d: %.0f", hc.itemTidx[r][t], double(hc.itemNs[r][t] - hc.roundNs[r]) * 1e-3);
            fprintf(stderr, "\n");
        }
    }
    int32_t err = 0;
    if (sync) TG_CUDA(cudaMemcpyAsync(&err, &W.ctx.ctrl->errFlag, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    TG_CUDA(cudaFreeAsync(W.base, st));
    W.base = nullptr;
    if (sync) {
        TG_CUDA(cudaStreamSynchronize(st));
        if (err) return fail(TG_ERR_CUDA, "solver reported internal error " + std::to_string(err));
    }
    return TG_OK;
}

}  // namespace

extern "C" {

const char* tg_last_error(void) { return g_err.c_str(); }
int32_t tg_version(void) { return 100; }

}  // extern "C"

namespace {

// Allocation, uploads and the validation kernel of one instance, all enqueued on the legacy default stream; the
// error word (device) is read by the caller after it has synchronised.
tg_status createAsync(int32_t L, int32_t K, int32_t P, int32_t m, const int32_t* time_us,
                      const int32_t* mem_mb, const int32_t* island_gpus, const int32_t* island_cap_mb,
                      const int32_t* bw_gbps, int32_t act_mb, tg_instance** out, int** dErrOut) {
    if (!time_us || !mem_mb || !island_gpus || !island_cap_mb || !bw_gbps || !out) return fail(TG_ERR_NULL, "NULL argument");
    if (L < 1 || L > TG_MAX_L || K < 1 || K > TG_MAX_K || P < 1 || P > TG_MAX_P || m < 1 || m > TG_MAX_M)
        return fail(TG_ERR_SHAPE, "L, K, P or m outside limits");
    if (act_mb < 0 || act_mb > (1 << 20)) return fail(TG_ERR_RANGE, "act_mb outside [0, 2^20]");
    int dev = 0;
    TG_CUDA(cudaGetDevice(&dev));
    DeviceState* D;
    tg_status s = deviceInit(dev, &D);
    if (s != TG_OK) return s;
    const int NS = L * (L + 1) / 2;
    const size_t nE = size_t(NS) * K * P;
    char* base = nullptr;
    Carver cv;
    const size_t oT = cv.take(nE * 4), oM = cv.take(nE * 4), oG = cv.take(K * 4), oC = cv.take(K * 4), oB = cv.take(K * K * 4), oE = cv.take(4);
    // stream-ordered allocation on the legacy default stream (pool-cached: no device synchronisation)
    TG_CUDA(poolAlloc(reinterpret_cast<void**>(&base), cv.off, 0));
    tg_instance* t = new (std::nothrow) tg_instance();
    if (!t) { cudaFreeAsync(base, 0); return fail(TG_ERR_OOM, "host allocation failed"); }
    t->L = L; t->K = K; t->P = P; t->m = m; t->act_mb = act_mb; t->NS = NS; t->device = dev;
    t->actmem = nullptr;
    t->xbound = 0;
    t->time_us = reinterpret_cast<int32_t*>(base + oT); t->mem_mb = reinterpret_cast<int32_t*>(base + oM);
    t->gpus = reinterpret_cast<int32_t*>(base + oG); t->cap_mb = reinterpret_cast<int32_t*>(base + oC);
    t->bw = reinterpret_cast<int32_t*>(base + oB);
    int* dErr = reinterpret_cast<int*>(base + oE);
    cudaError_t e = cudaMemcpyAsync(t->time_us, time_us, nE * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->mem_mb, mem_mb, nE * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->gpus, island_gpus, K * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->cap_mb, island_cap_mb, K * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->bw, bw_gbps, K * K * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemsetAsync(dErr, 0, 4, 0);
    if (e == cudaSuccess) {
        const int blocks = int(std::min<size_t>((nE + 255) / 256, 4096));
        tgValidateKernel<<<std::max(blocks, 1), 256>>>(t->time_us, t->mem_mb, t->gpus, t->cap_mb, t->bw, K, nE, dErr);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        cudaFreeAsync(base, 0);
        delete t;
        return fail(TG_ERR_CUDA, std::string("instance upload: ") + cudaGetErrorString(e));
    }
    *out = t;
    *dErrOut = dErr;
    return TG_OK;
}

tg_status rangeError(int herr, int index) {
    return fail(TG_ERR_RANGE, (index >= 0 ? "instance " + std::to_string(index) + ": " : std::string()) +
                                  "table value out of range (bits: 1 time, 2 mem, 4 bw, 8 gpus, 16 cap): " + std::to_string(herr));
}

}  // namespace

extern "C" {

tg_status tg_instance_create(int32_t L, int32_t K, int32_t P, int32_t m, const int32_t* time_us,
                             const int32_t* mem_mb, const int32_t* island_gpus, const int32_t* island_cap_mb,
                             const int32_t* bw_gbps, int32_t act_mb, tg_instance** out) {
    if (!out) return fail(TG_ERR_NULL, "NULL argument");
    tg_instance* t = nullptr;
    int* dErr = nullptr;
    tg_status s = createAsync(L, K, P, m, time_us, mem_mb, island_gpus, island_cap_mb, bw_gbps, act_mb, &t, &dErr);
    if (s != TG_OK) return s;
    int herr = 0;
    const cudaError_t e = cudaMemcpy(&herr, dErr, 4, cudaMemcpyDeviceToHost);   // the one synchronisation of the call
    if (e != cudaSuccess || herr) {
        tg_instance_destroy(t);
        if (e != cudaSuccess) return fail(TG_ERR_CUDA, std::string("instance upload: ") + cudaGetErrorString(e));
        return rangeError(herr, -1);
    }
    *out = t;
    return TG_OK;
}

tg_status tg_instance_create_classes(int32_t L, int32_t K, int32_t P, int32_t m, int32_t n_classes,
                                     const int32_t* class_of_slice, const int32_t* class_time_us,
                                     const int32_t* class_mem_mb, const int32_t* island_gpus,
                                     const int32_t* island_cap_mb, const int32_t* bw_gbps, int32_t act_mb, tg_instance** out) {
    if (!class_of_slice || !class_time_us || !class_mem_mb || !island_gpus || !island_cap_mb || !bw_gbps || !out)
        return fail(TG_ERR_NULL, "NULL argument");
    if (L < 1 || L > TG_MAX_L || K < 1 || K > TG_MAX_K || P < 1 || P > TG_MAX_P || m < 1 || m > TG_MAX_M)
        return fail(TG_ERR_SHAPE, "L, K, P or m outside limits");
    const int NS = L * (L + 1) / 2;
    if (n_classes < 1 || n_classes > NS) return fail(TG_ERR_SHAPE, "n_classes outside [1, NS]");
    if (act_mb < 0 || act_mb > (1 << 20)) return fail(TG_ERR_RANGE, "act_mb outside [0, 2^20]");
    int dev = 0;
    TG_CUDA(cudaGetDevice(&dev));
    DeviceState* D;
    tg_status s = deviceInit(dev, &D);
    if (s != TG_OK) return s;
    const size_t KP = size_t(K) * P, nE = size_t(NS) * KP, nC = size_t(n_classes) * KP;
    char *base = nullptr, *tmp = nullptr;
    Carver cv, ct;
    const size_t oT = cv.take(nE * 4), oM = cv.take(nE * 4), oG = cv.take(K * 4), oC = cv.take(K * 4), oB = cv.take(K * K * 4), oE = cv.take(4);
    // one block, kept by the instance: [classOf | class time | class mem], each 256-byte aligned (16-byte loads)
    const size_t oCls = ct.take(size_t(NS) * 4), oCt = ct.take(nC * 4), oCm = ct.take(nC * 4);
    TG_CUDA(poolAlloc(reinterpret_cast<void**>(&base), cv.off, 0));
    cudaError_t e = poolAlloc(reinterpret_cast<void**>(&tmp), ct.off, 0);
    if (e != cudaSuccess) { cudaFreeAsync(base, 0); return fail(TG_ERR_OOM, std::string("class tables: ") + cudaGetErrorString(e)); }
    tg_instance* t = new (std::nothrow) tg_instance();
    if (!t) { cudaFreeAsync(base, 0); cudaFreeAsync(tmp, 0); return fail(TG_ERR_OOM, "host allocation failed"); }
    t->L = L; t->K = K; t->P = P; t->m = m; t->act_mb = act_mb; t->NS = NS; t->device = dev;
    t->actmem = nullptr;
    t->xbound = 0;
    t->time_us = reinterpret_cast<int32_t*>(base + oT); t->mem_mb = reinterpret_cast<int32_t*>(base + oM);
    t->gpus = reinterpret_cast<int32_t*>(base + oG); t->cap_mb = reinterpret_cast<int32_t*>(base + oC);
    t->bw = reinterpret_cast<int32_t*>(base + oB);
    int* dErr = reinterpret_cast<int*>(base + oE);
    int32_t* dCls = reinterpret_cast<int32_t*>(tmp + oCls);
    int32_t* dCt = reinterpret_cast<int32_t*>(tmp + oCt);
    int32_t* dCm = reinterpret_cast<int32_t*>(tmp + oCm);
    e = cudaMemcpyAsync(dCls, class_of_slice, size_t(NS) * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dCt, class_time_us, nC * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dCm, class_mem_mb, nC * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->gpus, island_gpus, K * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->cap_mb, island_cap_mb, K * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->bw, bw_gbps, K * K * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemsetAsync(dErr, 0, 4, 0);
    int herr = 0;
    if (e == cudaSuccess) {
        const int blocks = std::max(1, int(std::min<size_t>((nE + 255) / 256, 4096)));
        tgExpandClassesKernel<<<blocks, 256>>>(dCls, dCt, dCm, n_classes, L, int(KP), nE, t->time_us, t->mem_mb, dErr);
        tgValidateKernel<<<blocks, 256>>>(t->time_us, t->mem_mb, t->gpus, t->cap_mb, t->bw, K, nE, dErr);
        e = cudaMemcpy(&herr, dErr, 4, cudaMemcpyDeviceToHost);   // the one synchronisation of the call
    }
    const bool toeplitz = !(herr & 64);   // bit 64 is not an error: the class of some slice depends on more than its length
    herr &= ~64;
    if (e != cudaSuccess || herr) {
        cudaFreeAsync(tmp, 0);
        tg_instance_destroy(t);
        if (e != cudaSuccess) return fail(TG_ERR_CUDA, std::string("instance upload: ") + cudaGetErrorString(e));
        return fail(TG_ERR_RANGE, "value out of range (bits: 1 time, 2 mem, 4 bw, 8 gpus, 16 cap, 32 class index): " + std::to_string(herr));
    }
    t->cls = reinterpret_cast<int32_t*>(tmp);
    t->nClasses = n_classes;
    t->toeplitz = toeplitz;
    *out = t;
    return TG_OK;
}

tg_status tg_instance_create_batch(int32_t n, const int32_t* L, const int32_t* K, const int32_t* P, const int32_t* m,
                                   const int32_t* const* time_us, const int32_t* const* mem_mb,
                                   const int32_t* const* island_gpus, const int32_t* const* island_cap_mb,
                                   const int32_t* const* bw_gbps, const int32_t* act_mb, tg_instance** out) {
    if (n < 0) return fail(TG_ERR_SHAPE, "n < 0");
    if (n == 0) return TG_OK;
    if (!L || !K || !P || !m || !time_us || !mem_mb || !island_gpus || !island_cap_mb || !bw_gbps || !act_mb || !out)
        return fail(TG_ERR_NULL, "NULL argument");
    for (int i = 0; i < n; ++i) out[i] = nullptr;
    for (int i = 0; i < n; ++i) {
        const std::string who = "instance " + std::to_string(i) + ": ";
        if (!time_us[i] || !mem_mb[i] || !island_gpus[i] || !island_cap_mb[i] || !bw_gbps[i]) return fail(TG_ERR_NULL, who + "NULL argument");
        if (L[i] < 1 || L[i] > TG_MAX_L || K[i] < 1 || K[i] > TG_MAX_K || P[i] < 1 || P[i] > TG_MAX_P || m[i] < 1 || m[i] > TG_MAX_M)
            return fail(TG_ERR_SHAPE, who + "L, K, P or m outside limits");
        if (act_mb[i] < 0 || act_mb[i] > (1 << 20)) return fail(TG_ERR_RANGE, who + "act_mb outside [0, 2^20]");
    }
    int dev = 0;
    TG_CUDA(cudaGetDevice(&dev));
    DeviceState* D;
    tg_status s = deviceInit(dev, &D);
    if (s != TG_OK) return s;

    // One allocation for the batch: [per instance: time, mem] [small arrays of all instances] [descriptors] [error words].
    // A handful of driver calls per instance (two table uploads) instead of eight, one validation launch, one
    // synchronisation.
    Carver cv;
    const size_t nn = size_t(n);
    std::vector<size_t> oT(nn), oM(nn), oS(nn);
    size_t smallInts = 0, maxE = 0;
    for (int i = 0; i < n; ++i) {
        const size_t nE = size_t(L[i]) * (L[i] + 1) / 2 * K[i] * P[i];
        oT[size_t(i)] = cv.take(nE * 4);
        oM[size_t(i)] = cv.take(nE * 4);
        oS[size_t(i)] = smallInts;                       // gpus[K], cap[K], bw[K*K]
        smallInts += size_t(K[i]) * (2 + K[i]);
        maxE = std::max(maxE, nE);
    }
    const size_t oSmall = cv.take(smallInts * 4), oDesc = cv.take(sizeof(TgValidateDesc) * size_t(n)), oErr = cv.take(size_t(n) * 4);
    TgBatchBlock* blk = new (std::nothrow) TgBatchBlock();
    if (!blk) return fail(TG_ERR_OOM, "host allocation failed");
    cudaError_t e = poolAlloc(reinterpret_cast<void**>(&blk->base), cv.off, 0);
    if (e != cudaSuccess) {
        delete blk;
        cudaGetLastError();
        return fail(e == cudaErrorMemoryAllocation ? TG_ERR_OOM : TG_ERR_CUDA, std::string("batch allocation: ") + cudaGetErrorString(e));
    }
    char* base = blk->base;
    {   // the upload streams start behind the allocation (stream-ordered on the legacy default stream)
        std::lock_guard<std::mutex> lk(g_mu);   // one batch at a time uses the upload streams and their events
        e = cudaEventRecord(D->upEv[4], 0);
        for (int q = 0; q < 4 && e == cudaSuccess; ++q) e = cudaStreamWaitEvent(D->up[q], D->upEv[4], 0);
    }
    if (e != cudaSuccess) { cudaFreeAsync(blk->base, 0); delete blk; cudaGetLastError(); return fail(TG_ERR_CUDA, "batch upload: stream setup"); }
    int32_t* dSmall = reinterpret_cast<int32_t*>(base + oSmall);
    std::vector<int32_t> hSmall(smallInts);
    std::vector<TgValidateDesc> hDesc(nn);
    struct Late { const int32_t* src; int32_t* dst; size_t ints; };
    std::vector<Late> late;                              // small arrays that live in device memory: copied after the staged ones
    int made = 0;
    for (; made < n && e == cudaSuccess; ++made) {
        const int i = made;
        tg_instance* t = new (std::nothrow) tg_instance();
        if (!t) { e = cudaErrorMemoryAllocation; break; }
        const int Ki = K[i];
        const size_t nE = size_t(L[i]) * (L[i] + 1) / 2 * Ki * P[i];
        t->block = blk;
        blk->refs.fetch_add(1);
        t->L = L[i]; t->K = Ki; t->P = P[i]; t->m = m[i]; t->act_mb = act_mb[i]; t->NS = L[i] * (L[i] + 1) / 2; t->device = dev;
        t->actmem = nullptr;
        t->xbound = 0;
        t->time_us = reinterpret_cast<int32_t*>(base + oT[size_t(i)]);
        t->mem_mb = reinterpret_cast<int32_t*>(base + oM[size_t(i)]);
        t->gpus = dSmall + oS[size_t(i)];
        t->cap_mb = t->gpus + Ki;
        t->bw = t->cap_mb + Ki;
        out[i] = t;
        // the table uploads are dealt to four streams: a single stream moved 188 KB tables at a third of the link's
        // rate (every copy waits for the previous one's completion before it starts)
        e = cudaMemcpyAsync(t->time_us, time_us[i], nE * 4, cudaMemcpyDefault, D->up[(2 * i) & 3]);
        if (e == cudaSuccess) e = cudaMemcpyAsync(t->mem_mb, mem_mb[i], nE * 4, cudaMemcpyDefault, D->up[(2 * i + 1) & 3]);
        const int32_t* srcs[3] = {island_gpus[i], island_cap_mb[i], bw_gbps[i]};
        int32_t* dsts[3] = {t->gpus, t->cap_mb, t->bw};
        const size_t lens[3] = {size_t(Ki), size_t(Ki), size_t(Ki) * Ki};
        for (int q = 0; q < 3; ++q) {
            int32_t* hdst = hSmall.data() + (dsts[q] - dSmall);
            if (isDevicePtr(srcs[q])) { late.push_back({srcs[q], dsts[q], lens[q]}); memset(hdst, 0, lens[q] * 4); }
            else memcpy(hdst, srcs[q], lens[q] * 4);
        }
        hDesc[size_t(i)] = TgValidateDesc{t->time_us, t->mem_mb, t->gpus, t->cap_mb, t->bw, Ki, (unsigned long long)nE};
    }
    int* dErr = reinterpret_cast<int*>(base + oErr);
    std::vector<int> herr(nn, 0);
    for (int q = 0; q < 4; ++q) {   // the validation (default stream) runs behind every upload, also on the error paths
        cudaError_t e2 = cudaEventRecord(D->upEv[q], D->up[q]);
        if (e2 == cudaSuccess) e2 = cudaStreamWaitEvent(0, D->upEv[q], 0);
        if (e == cudaSuccess) e = e2;
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(dSmall, hSmall.data(), smallInts * 4, cudaMemcpyHostToDevice, 0);
    for (size_t q = 0; q < late.size() && e == cudaSuccess; ++q)
        e = cudaMemcpyAsync(late[q].dst, late[q].src, late[q].ints * 4, cudaMemcpyDeviceToDevice, 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(base + oDesc, hDesc.data(), sizeof(TgValidateDesc) * size_t(n), cudaMemcpyHostToDevice, 0);
    if (e == cudaSuccess) e = cudaMemsetAsync(dErr, 0, size_t(n) * 4, 0);
    if (e == cudaSuccess) {
        const int bx = int(std::max<size_t>(1, std::min<size_t>((maxE + 255) / 256, 64)));
        for (int y0 = 0; y0 < n && e == cudaSuccess; y0 += 65535) {      // gridDim.y limit
            const int ny = std::min(n - y0, 65535);
            tgValidateBatchKernel<<<dim3(bx, ny), 256>>>(reinterpret_cast<const TgValidateDesc*>(base + oDesc) + y0, dErr + y0);
            e = cudaGetLastError();
        }
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(herr.data(), dErr, size_t(n) * 4, cudaMemcpyDeviceToHost, 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);   // the one synchronisation of the call
    std::string err;
    if (e != cudaSuccess) {
        s = e == cudaErrorMemoryAllocation ? TG_ERR_OOM : TG_ERR_CUDA;
        err = std::string("batch upload: ") + cudaGetErrorString(e);
        cudaGetLastError();
    } else {
        for (int i = 0; i < n && s == TG_OK; ++i)
            if (herr[size_t(i)]) { s = rangeError(herr[size_t(i)], i); err = g_err; }
    }
    if (s != TG_OK) {   // all or nothing
        bool any = false;
        for (int i = 0; i < n; ++i) if (out[i]) { any = true; tg_instance_destroy(out[i]); out[i] = nullptr; }
        if (!any) { cudaFreeAsync(blk->base, 0); delete blk; }
        return fail(s, err);
    }
    return TG_OK;
}

tg_status tg_instance_destroy(tg_instance* inst) {
    if (!inst) return TG_OK;
    if (inst->actmem) cudaFreeAsync(inst->actmem, 0);
    if (inst->slow) cudaFreeAsync(inst->slow, 0);
    if (inst->cls) cudaFreeAsync(inst->cls, 0);
    if (inst->block) {   // created by tg_instance_create_batch: the allocation goes with the last instance of the batch
        TgBatchBlock* blk = inst->block;
        if (blk->refs.fetch_sub(1) == 1) { cudaFreeAsync(blk->base, 0); delete blk; }
    } else {
        cudaFreeAsync(inst->time_us, 0);  // base of the single allocation
    }
    delete inst;
    return TG_OK;
}

tg_status tg_instance_set_actmem(tg_instance* inst, const int32_t* actmem_mb) {
    if (!inst) return fail(TG_ERR_NULL, "inst is NULL");
    if (inst->actmem) { cudaFreeAsync(inst->actmem, 0); inst->actmem = nullptr; }
    if (!actmem_mb) return TG_OK;
    if (inst->cls) { cudaFreeAsync(inst->cls, 0); inst->cls = nullptr; }   // (from here on the expanded tables are the instance)
    if (inst->slow) return fail(TG_ERR_SHAPE, "the instance has multi-stage partial plans (tg_instance_set_stages): the combination with a footprint table is not built");
    const size_t nE = size_t(inst->NS) * inst->K * inst->P;
    int32_t* d = nullptr;
    TG_CUDA(poolAlloc(reinterpret_cast<void**>(&d), nE * 4 + 4, 0));
    int* dErr = reinterpret_cast<int*>(d + nE);
    cudaError_t e = cudaMemcpyAsync(d, actmem_mb, nE * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = cudaMemsetAsync(dErr, 0, 4, 0);
    int herr = 0;
    if (e == cudaSuccess) {
        const int blocks = int(std::min<size_t>((nE + 255) / 256, 4096));
        tgValidateNonNegKernel<<<std::max(blocks, 1), 256>>>(d, nE, dErr);
        e = cudaMemcpy(&herr, dErr, 4, cudaMemcpyDeviceToHost);
    }
    if (e != cudaSuccess || herr) {
        cudaFreeAsync(d, 0);
        if (e != cudaSuccess) return fail(TG_ERR_CUDA, std::string("actmem upload: ") + cudaGetErrorString(e));
        return fail(TG_ERR_RANGE, "actmem_mb must be in [0, 2^20]");
    }
    inst->actmem = d;
    return TG_OK;
}

tg_status tg_instance_set_stages(tg_instance* inst, const int32_t* slow_us, const int32_t* n_stages) {
    if (!inst) return fail(TG_ERR_NULL, "inst is NULL");
    if (inst->slow) { cudaFreeAsync(inst->slow, 0); inst->slow = nullptr; inst->qst = nullptr; }
    if (!slow_us) return TG_OK;
    if (inst->cls) { cudaFreeAsync(inst->cls, 0); inst->cls = nullptr; }   // (from here on the expanded tables are the instance)
    if (inst->actmem) return fail(TG_ERR_SHAPE, "the instance has a footprint table (tg_instance_set_actmem): the combination with multi-stage partial plans is not built");
    if (inst->nAct) return fail(TG_ERR_SHAPE, "the instance has per-boundary activation sizes (tg_instance_set_boundary_act): the combination with multi-stage partial plans is not built");
    const size_t nE = size_t(inst->NS) * inst->K * inst->P;
    int32_t* d = nullptr;
    TG_CUDA(poolAlloc(reinterpret_cast<void**>(&d), 2 * nE * 4 + 4, 0));
    int32_t* dq = d + nE;
    int* dErr = reinterpret_cast<int*>(d + 2 * nE);
    cudaError_t e = cudaMemcpyAsync(d, slow_us, nE * 4, cudaMemcpyDefault, 0);
    if (e == cudaSuccess) e = n_stages ? cudaMemcpyAsync(dq, n_stages, nE * 4, cudaMemcpyDefault, 0) : cudaSuccess;
    if (e == cudaSuccess) e = cudaMemsetAsync(dErr, 0, 4, 0);
    int herr = 0;
    if (e == cudaSuccess) {
        const int blocks = int(std::min<size_t>((nE + 255) / 256, 4096));
        tgValidateStagesKernel<<<std::max(blocks, 1), 256>>>(inst->time_us, d, dq, n_stages != nullptr, nE, dErr);
        e = cudaMemcpy(&herr, dErr, 4, cudaMemcpyDeviceToHost);
    }
    if (e != cudaSuccess || herr) {
        cudaFreeAsync(d, 0);
        if (e != cudaSuccess) return fail(TG_ERR_CUDA, std::string("stage tables upload: ") + cudaGetErrorString(e));
        return fail(TG_ERR_RANGE, "slow_us must be in [0, time_us] on every valid entry and n_stages in [1, 255]");
    }
    inst->slow = d;
    inst->qst = dq;
    return TG_OK;
}

tg_status tg_plan_pipeline_stages(tg_instance* inst, const tg_result* result, int32_t* n_out) {
    if (!inst || !result || !n_out) return fail(TG_ERR_NULL, "NULL argument");
    const int n = result->n_stages;
    if (n < 0 || n > TG_MAX_K) return fail(TG_ERR_RANGE, "result.n_stages outside [0, TG_MAX_K]");
    int total = 0;
    for (int i = 0; i < n; ++i) {
        const int a = result->stage_begin[i], b = i + 1 < n ? result->stage_begin[i + 1] : inst->L;
        const int k = result->stage_island[i], p = result->stage_plan[i];
        if (a < 0 || b <= a || b > inst->L || k < 0 || k >= inst->K || p < 0 || p >= inst->P) return fail(TG_ERR_RANGE, "result does not describe a plan of this instance");
        int q = 1;
        if (inst->qst) TG_CUDA(cudaMemcpy(&q, inst->qst + (size_t(tgSliceIdx(inst->L, a, b)) * inst->K + k) * inst->P + p, 4, cudaMemcpyDeviceToHost));
        total += q;
    }
    *n_out = total;
    return TG_OK;
}

tg_status tg_instance_set_boundary_act(tg_instance* inst, const int32_t* act_mb_b) {
    if (!inst) return fail(TG_ERR_NULL, "inst is NULL");
    if (!act_mb_b) { inst->nAct = 0; return TG_OK; }
    if (inst->slow) return fail(TG_ERR_SHAPE, "the instance has multi-stage partial plans (tg_instance_set_stages): the combination with per-boundary activation sizes is not built");
    const int L = inst->L;
    std::vector<int32_t> h(size_t(L) + 1);
    TG_CUDA(cudaMemcpy(h.data(), act_mb_b, (size_t(L) + 1) * 4, cudaMemcpyDefault));
    int nAct = 0;
    int32_t vals[TG_MAX_ACT];
    uint8_t cls[256];
    memset(cls, 0, sizeof(cls));
    for (int b = 1; b < L; ++b) {
        if (h[b] < 0 || h[b] > (1 << 20)) return fail(TG_ERR_RANGE, "act_mb_b[" + std::to_string(b) + "] outside [0, 2^20]");
        int c = 0;
        while (c < nAct && vals[c] != h[b]) ++c;
        if (c == nAct) {
            if (nAct == TG_MAX_ACT) return fail(TG_ERR_SHAPE, "more than TG_MAX_ACT distinct activation sizes");
            vals[nAct++] = h[b];
        }
        cls[b] = uint8_t(c);
    }
    if (nAct == 0) { vals[0] = 0; nAct = 1; }            // a one-layer model has no boundary
    inst->nAct = nAct;
    memset(inst->actVal, 0, sizeof(inst->actVal));
    memcpy(inst->actVal, vals, size_t(nAct) * 4);
    memcpy(inst->clsOf, cls, sizeof(cls));
    return TG_OK;
}

tg_status tg_instance_set_transfer_bound(tg_instance* inst, int32_t on) {
    if (!inst) return fail(TG_ERR_NULL, "inst is NULL");
    inst->xbound = on ? 1 : 0;
    return TG_OK;
}

tg_status tg_solve_batch_ex(tg_instance* const* instances, int32_t n, tg_result* out, uint32_t flags,
                            tg_solve_stats* stats, void* cuda_stream) {
    if (n == 0) return TG_OK;
    if (!out) return fail(TG_ERR_NULL, "out is NULL");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Workspace W;
    tg_status s = prepare(instances, n, true, st, W);
    if (s != TG_OK) return s;
    W.ctx.out = W.outDev; W.ctx.flags = flags; W.ctx.mode = 0;
    s = launchSolve(W, st);
    if (s != TG_OK) return s;
    return finish(W, n, out, stats, st);
}

tg_status tg_solve_batch(tg_instance* const* instances, int32_t n, tg_result* out, void* cuda_stream) {
    return tg_solve_batch_ex(instances, n, out, TG_SOLVE_DEFAULT, nullptr, cuda_stream);
}

tg_status tg_dp_at(tg_instance* inst, int64_t T, tg_result* out, void* cuda_stream) {
    if (!inst || !out) return fail(TG_ERR_NULL, "NULL argument");
    if (T > TG_TIME_MAX) T = -1;  // every finite cost is admissible
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Workspace W;
    tg_instance* arr[1] = {inst};
    tg_status s = prepare(arr, 1, true, st, W);
    if (s != TG_OK) return s;
    W.ctx.out = W.outDev; W.ctx.flags = 0; W.ctx.mode = 1;
    W.ctx.dpT = T < 0 ? TG_TINF : uint32_t(T);
    s = launchSolve(W, st);
    if (s != TG_OK) return s;
    return finish(W, 1, out, nullptr, st);
}

// steps 1-3 for one instance; cand_out receives at most cand_capacity thresholds, *n_cand_out the full count
static tg_status reduceImpl(tg_instance* inst, int32_t* c_out, int32_t* argp_out, int32_t* x_out, int32_t* cand_out,
                            int64_t cand_capacity, int32_t* n_cand_out, void* cuda_stream) {
    if (!inst) return fail(TG_ERR_NULL, "inst is NULL");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Workspace W;
    tg_instance* arr[1] = {inst};
    tg_status s = prepare(arr, 1, false, st, W);
    if (s != TG_OK) return s;
    const int cells = inst->NS * inst->K, K = inst->K;
    int32_t *dc = nullptr, *da = nullptr, *dx = nullptr;
    cudaError_t e = poolAlloc(reinterpret_cast<void**>(&dc), size_t(cells) * 4 * 2 + K * K * 4, st);
    TgInstDev hI;
    if (e == cudaSuccess) {
        da = dc + cells; dx = da + cells;
        tgExportKernel<<<std::max(1, std::min((cells + 255) / 256, 1024)), 256, 0, st>>>(W.inst, dc, da, dx);
        e = cudaMemcpyAsync(&hI, W.inst, sizeof(TgInstDev), cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess && c_out) e = cudaMemcpyAsync(c_out, dc, size_t(cells) * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && argp_out) e = cudaMemcpyAsync(argp_out, da, size_t(cells) * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && x_out) e = cudaMemcpyAsync(x_out, dx, size_t(K) * K * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && cand_out && hI.ncand > 0 && cand_capacity > 0)
        e = cudaMemcpyAsync(cand_out, hI.cand, size_t(std::min<int64_t>(hI.ncand, cand_capacity)) * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (dc) cudaFreeAsync(dc, st);
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? TG_ERR_OOM : TG_ERR_CUDA, std::string("tg_reduce: ") + cudaGetErrorString(e));
    if (n_cand_out) *n_cand_out = hI.ncand;
    return TG_OK;
}

tg_status tg_reduce(tg_instance* inst, int32_t* c_out, int32_t* argp_out, int32_t* x_out, int32_t* cand_out,
                    int32_t* n_cand_out, void* cuda_stream) {
    if (!inst) return fail(TG_ERR_NULL, "inst is NULL");
    return reduceImpl(inst, c_out, argp_out, x_out, cand_out, int64_t(inst->NS) * inst->K, n_cand_out, cuda_stream);
}

tg_status tg_candidates(tg_instance* inst, int32_t* cand_out, int64_t capacity, int32_t* n_cand_out, void* cuda_stream) {
    if (!inst || !n_cand_out) return fail(TG_ERR_NULL, "NULL argument");
    if (capacity < 0 || (capacity > 0 && !cand_out)) return fail(TG_ERR_RANGE, "capacity < 0, or capacity > 0 without a buffer");
    return reduceImpl(inst, nullptr, nullptr, nullptr, cand_out, capacity, n_cand_out, cuda_stream);
}

tg_status tg_prune_batch(tg_instance* const* instances, int32_t n, tg_prune_mode mode, int64_t threshold, int64_t* counts_out,
                         void* cuda_stream) {
    if (n == 0) return TG_OK;
    if (!instances || !counts_out) return fail(TG_ERR_NULL, "NULL argument");
    if (n < 0 || n > 65535) return fail(TG_ERR_SHAPE, "n must be in [0, 65535]");
    if (mode != TG_PRUNE_EXACT && mode != TG_PRUNE_IMBALANCE && mode != TG_PRUNE_BOTTLENECK)
        return fail(TG_ERR_RANGE, "unknown prune mode");
    if (mode == TG_PRUNE_IMBALANCE && (threshold < 1000 || threshold > 16384))
        return fail(TG_ERR_RANGE, "theta must be in [1000, 16384] permille");
    if (mode == TG_PRUNE_BOTTLENECK && threshold < 0) return fail(TG_ERR_RANGE, "bottleneck cap must be >= 0");
    std::vector<TgPruneDesc> h(n);
    int maxCells = 0;
    for (int i = 0; i < n; ++i) {
        tg_instance* t = instances[i];
        if (!t) return fail(TG_ERR_NULL, "instances[" + std::to_string(i) + "] is NULL");
        if (t->slow) return fail(TG_ERR_SHAPE, "instances[" + std::to_string(i) + "] has multi-stage partial plans: tg_prune is not built for them");
        if (t->cls) { cudaFreeAsync(t->cls, 0); t->cls = nullptr; }   // pruning edits the expanded tables: they are the instance from now on
        h[i] = TgPruneDesc{t->time_us, t->mem_mb, t->actmem, t->cap_mb, t->L, t->K, t->P, t->NS * t->K};
        maxCells = std::max(maxCells, h[i].nCells);
    }
    {   // an instance listed twice would be pruned by two grids at once
        std::vector<const tg_instance*> seen(instances, instances + n);
        std::sort(seen.begin(), seen.end());
        if (std::adjacent_find(seen.begin(), seen.end()) != seen.end()) return fail(TG_ERR_RANGE, "an instance appears twice in the batch");
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t oCounts = 0, oCap = size_t(n) * 32, oDesc = oCap + size_t(n) * (TG_MAX_K + 1) * 8;
    char* ws = nullptr;
    TG_CUDA(poolAlloc(reinterpret_cast<void**>(&ws), oDesc + sizeof(TgPruneDesc) * size_t(n), st));
    unsigned long long* dCounts = reinterpret_cast<unsigned long long*>(ws + oCounts);
    long long* dCap = reinterpret_cast<long long*>(ws + oCap);
    TgPruneDesc* dDesc = reinterpret_cast<TgPruneDesc*>(ws + oDesc);
    TG_CUDA(cudaMemsetAsync(ws, 0, oCap, st));
    TG_CUDA(cudaMemcpyAsync(dDesc, h.data(), sizeof(TgPruneDesc) * size_t(n), cudaMemcpyHostToDevice, st));
    const dim3 g((maxCells + 255) / 256, n), g1((maxCells + TG_PR_NT - 1) / TG_PR_NT, n);
    {   // cell pass: the register path is compiled for P = 4 and P = 8 (picked from the first instance); TG_PR_U cells per
        // thread (two of P = 8) once that still leaves every SM a few CTAs
        DeviceState* DS = nullptr;
        int dev = 0;
        TG_CUDA(cudaGetDevice(&dev));
        const tg_status sd = deviceInit(dev, &DS);
        if (sd != TG_OK) { cudaFreeAsync(ws, st); return sd; }
        const int P0 = instances[0]->P;
        const dim3 g2((maxCells + 2 * TG_PR_NT - 1) / (2 * TG_PR_NT), n);
        const dim3 gU((maxCells + TG_PR_U * TG_PR_NT - 1) / (TG_PR_U * TG_PR_NT), n);
        const bool wide = int64_t(g2.x) * n >= 4 * DS->numSMs;   // (several cells a thread once that still leaves every SM a few CTAs)
        bool act = false;
        for (int i = 0; i < n; ++i) act = act || instances[i]->actmem != nullptr;
#define TG_PRUNE_LAUNCH(PV, U, G) \
        do { if (act) tgPruneCellKernel<PV, U, true><<<G, TG_PR_NT, 0, st>>>(dDesc, int(mode), threshold, dCounts); \
             else tgPruneCellKernel<PV, U, false><<<G, TG_PR_NT, 0, st>>>(dDesc, int(mode), threshold, dCounts); } while (0)
        if (P0 == 4) {
            if (wide) TG_PRUNE_LAUNCH(1, TG_PR_U, gU); else TG_PRUNE_LAUNCH(1, 1, g1);
        } else if (P0 == 8) {
            if (wide) TG_PRUNE_LAUNCH(2, 2, g2); else TG_PRUNE_LAUNCH(2, 1, g1);
        } else {
            TG_PRUNE_LAUNCH(0, 1, g1);
        }
#undef TG_PRUNE_LAUNCH
    }
    if (mode == TG_PRUNE_IMBALANCE) {
        tgPruneTauKernel<<<n, 256, 0, st>>>(dDesc, dCap);
        tgPruneImbalanceKernel<<<g, 256, 0, st>>>(dDesc, dCap, threshold, dCounts);
    }
    TG_CUDA(cudaGetLastError());
    std::vector<unsigned long long> hc(size_t(n) * 4);
    TG_CUDA(cudaMemcpyAsync(hc.data(), dCounts, size_t(n) * 32, cudaMemcpyDeviceToHost, st));
    TG_CUDA(cudaStreamSynchronize(st));   // also keeps h alive until the descriptor upload has been read
    TG_CUDA(cudaFreeAsync(ws, st));
    for (size_t i = 0; i < size_t(n) * 4; ++i) counts_out[i] = int64_t(hc[i]);
    return TG_OK;
}

tg_status tg_prune(tg_instance* inst, tg_prune_mode mode, int64_t threshold, int64_t counts_out[4], void* cuda_stream) {
    if (!inst || !counts_out) return fail(TG_ERR_NULL, "NULL argument");
    return tg_prune_batch(&inst, 1, mode, threshold, counts_out, cuda_stream);
}

// ---------------------------------------------------------------------------------------------
// tg_prune_batch_static: tg_prune_batch for callers that must not allocate device memory (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  The pass's scratch -- the per-rule counters, the R3 caps and
// the instance descriptors the kernels read -- lives in ONE file-scope device array of fixed size; every GPU that loads
// the library holds it until exit.  The kernels are the ones tg_prune_batch launches, unchanged.
// ---------------------------------------------------------------------------------------------
constexpr size_t TG_PS_COUNTS = size_t(TG_PRUNE_STATIC_MAX_N) * 32;                       // [n][4] unsigned long long
constexpr size_t TG_PS_CAP = size_t(TG_PRUNE_STATIC_MAX_N) * (TG_MAX_K + 1) * 8;          // [n][TG_MAX_K + 1] long long (R3)
constexpr size_t TG_PS_DESC = size_t(TG_PRUNE_STATIC_MAX_N) * sizeof(TgPruneDesc);
constexpr size_t TG_PS_BYTES = TG_PS_COUNTS + TG_PS_CAP + TG_PS_DESC;                     // 221 184 bytes
static_assert(TG_PS_COUNTS % 256 == 0 && TG_PS_CAP % 256 == 0, "parts of the static scratch keep the 256-byte alignment");
static_assert(TG_PS_BYTES <= (256u << 10), "static prune scratch: stated maximum is 256 KB");
static __device__ __align__(256) unsigned char tgPruneStaticScratch[TG_PS_BYTES];

struct StaticPruneState {
    bool ready = false;
    unsigned char* scratch = nullptr;   // DEVICE address of tgPruneStaticScratch on this device (the symbol itself is a host-side stand-in)
    int numSMs = 0;
};
StaticPruneState g_staticPrune[64];
std::mutex g_staticPruneMu;   // set-up, and the host-side descriptor staging below

tg_status tg_prune_batch_static(tg_instance* const* instances, int32_t n, tg_prune_mode mode, int64_t threshold, int64_t* counts_out,
                                void* cuda_stream) {
    if (n == 0) return TG_OK;
    if (!instances || !counts_out) return fail(TG_ERR_NULL, "NULL argument");
    if (n < 0 || n > TG_PRUNE_STATIC_MAX_N)
        return fail(TG_ERR_SHAPE, "tg_prune_batch_static: n = " + std::to_string(n) + " outside [0, TG_PRUNE_STATIC_MAX_N = " +
                                      std::to_string(TG_PRUNE_STATIC_MAX_N) + "]: the static scratch holds no more; use tg_prune_batch");
    if (mode != TG_PRUNE_EXACT && mode != TG_PRUNE_IMBALANCE && mode != TG_PRUNE_BOTTLENECK)
        return fail(TG_ERR_RANGE, "unknown prune mode");
    if (mode == TG_PRUNE_IMBALANCE && (threshold < 1000 || threshold > 16384))
        return fail(TG_ERR_RANGE, "theta must be in [1000, 16384] permille");
    if (mode == TG_PRUNE_BOTTLENECK && threshold < 0) return fail(TG_ERR_RANGE, "bottleneck cap must be >= 0");
    int dev = 0;
    TG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(TG_ERR_CUDA, "device ordinal out of range");
    std::lock_guard<std::mutex> lk(g_staticPruneMu);
    static TgPruneDesc h[TG_PRUNE_STATIC_MAX_N];            // host staging, fixed size (under the mutex)
    static const tg_instance* seen[TG_PRUNE_STATIC_MAX_N];
    int maxCells = 0;
    bool act = false;
    for (int i = 0; i < n; ++i) {
        tg_instance* t = instances[i];
        if (!t) return fail(TG_ERR_NULL, "instances[" + std::to_string(i) + "] is NULL");
        if (t->device != dev) return fail(TG_ERR_CUDA, "instance was created on another device");
        if (t->slow) return fail(TG_ERR_SHAPE, "instances[" + std::to_string(i) + "] has multi-stage partial plans: tg_prune is not built for them");
        if (t->cls) return fail(TG_ERR_SHAPE, "instances[" + std::to_string(i) + "] keeps class tables: pruning would have to free them; use tg_prune_batch");
        h[i] = TgPruneDesc{t->time_us, t->mem_mb, t->actmem, t->cap_mb, t->L, t->K, t->P, t->NS * t->K};
        maxCells = std::max(maxCells, h[i].nCells);
        act = act || t->actmem != nullptr;
        seen[i] = t;
    }
    std::sort(seen, seen + n);
    if (std::adjacent_find(seen, seen + n) != seen + n) return fail(TG_ERR_RANGE, "an instance appears twice in the batch");
    StaticPruneState& S = g_staticPrune[dev];
    if (!S.ready) {   // once per device, with that device current: the array's device address; nothing is allocated
        void* ptr = nullptr;
        TG_CUDA(cudaGetSymbolAddress(&ptr, tgPruneStaticScratch));
        if (!ptr) return fail(TG_ERR_CUDA, "cudaGetSymbolAddress returned NULL for the static scratch");
        TG_CUDA(cudaDeviceGetAttribute(&S.numSMs, cudaDevAttrMultiProcessorCount, dev));
        S.scratch = static_cast<unsigned char*>(ptr);
        S.ready = true;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned long long* dCounts = reinterpret_cast<unsigned long long*>(S.scratch);
    long long* dCap = reinterpret_cast<long long*>(S.scratch + TG_PS_COUNTS);
    TgPruneDesc* dDesc = reinterpret_cast<TgPruneDesc*>(S.scratch + TG_PS_COUNTS + TG_PS_CAP);
    // the array keeps the last call's contents: counters and caps start at zero, the descriptors are overwritten
    TG_CUDA(cudaMemsetAsync(S.scratch, 0, TG_PS_COUNTS + TG_PS_CAP, st));
    TG_CUDA(cudaMemcpyAsync(dDesc, h, sizeof(TgPruneDesc) * size_t(n), cudaMemcpyHostToDevice, st));
    const dim3 g((maxCells + 255) / 256, n), g1((maxCells + TG_PR_NT - 1) / TG_PR_NT, n), g2((maxCells + 2 * TG_PR_NT - 1) / (2 * TG_PR_NT), n),
               gU((maxCells + TG_PR_U * TG_PR_NT - 1) / (TG_PR_U * TG_PR_NT), n);
    const bool wide = int64_t(g2.x) * n >= 4 * S.numSMs;
    const int P0 = instances[0]->P;
#define TG_PRUNE_LAUNCH(PV, U, G) \
    do { if (act) tgPruneCellKernel<PV, U, true><<<G, TG_PR_NT, 0, st>>>(dDesc, int(mode), threshold, dCounts); \
         else tgPruneCellKernel<PV, U, false><<<G, TG_PR_NT, 0, st>>>(dDesc, int(mode), threshold, dCounts); } while (0)
    if (P0 == 4) {
        if (wide) TG_PRUNE_LAUNCH(1, TG_PR_U, gU); else TG_PRUNE_LAUNCH(1, 1, g1);
    } else if (P0 == 8) {
        if (wide) TG_PRUNE_LAUNCH(2, 2, g2); else TG_PRUNE_LAUNCH(2, 1, g1);
    } else {
        TG_PRUNE_LAUNCH(0, 1, g1);
    }
#undef TG_PRUNE_LAUNCH
    if (mode == TG_PRUNE_IMBALANCE) {
        tgPruneTauKernel<<<n, 256, 0, st>>>(dDesc, dCap);
        tgPruneImbalanceKernel<<<g, 256, 0, st>>>(dDesc, dCap, threshold, dCounts);
    }
    TG_CUDA(cudaGetLastError());
    static_assert(sizeof(unsigned long long) == sizeof(int64_t), "counts are copied as they are");
    TG_CUDA(cudaMemcpyAsync(counts_out, dCounts, size_t(n) * 32, cudaMemcpyDeviceToHost, st));
    TG_CUDA(cudaStreamSynchronize(st));   // counts_out is valid; the host staging and the scratch are free for the next call
    return TG_OK;
}

tg_status tg_islands_build(int32_t n_nodes, const int32_t* node_gpus, const int32_t* node_compute, const int32_t* node_mem_mb,
                           const int32_t* node_intra_bw, const int32_t* inter_bw, int32_t eps_c, int32_t eps_m, int32_t eps_i,
                           int32_t* island_of_node, int32_t* k_out, int32_t* island_gpus, int32_t* island_cap_mb, int32_t* bw_gbps) {
    if (!node_gpus || !node_compute || !node_mem_mb || !node_intra_bw || !inter_bw || !island_of_node || !k_out || !island_gpus ||
        !island_cap_mb || !bw_gbps)
        return fail(TG_ERR_NULL, "NULL argument");
    if (n_nodes < 1 || n_nodes > TG_MAX_NODES) return fail(TG_ERR_SHAPE, "n_nodes outside [1, TG_MAX_NODES]");
    if (eps_c < 0 || eps_m < 0 || eps_i < 0 || eps_c > 1000000 || eps_m > 1000000 || eps_i > 1000000)
        return fail(TG_ERR_RANGE, "tolerances must be in [0, 10^6] permille");
    const int N = n_nodes;
    for (int n = 0; n < N; ++n) {
        if (node_gpus[n] < 1 || node_compute[n] < 1 || node_mem_mb[n] < 0 || node_intra_bw[n] < 1)
            return fail(TG_ERR_RANGE, "node " + std::to_string(n) + ": gpus, compute and intra-node bandwidth must be >= 1, memory >= 0");
        if (node_gpus[n] > (1 << 20) || node_compute[n] > (1 << 20) || node_intra_bw[n] > (1 << 20))
            return fail(TG_ERR_RANGE, "node " + std::to_string(n) + ": value above 2^20");
        for (int m = 0; m < N; ++m)
            if (m != n && (inter_bw[size_t(n) * N + m] < 1 || inter_bw[size_t(n) * N + m] > (1 << 20)))
                return fail(TG_ERR_RANGE, "inter_bw must be in [1, 2^20] off the diagonal");
    }
    int dev = 0;
    TG_CUDA(cudaGetDevice(&dev));
    DeviceState* D;
    tg_status st = deviceInit(dev, &D);
    if (st != TG_OK) return st;
    // one device buffer: [gpus | comp | mem | intra | inter | islandOf | K | islandGpus | islandCap | bw]
    const size_t nIn = size_t(4) * N + size_t(N) * N, nOut = size_t(N) + 1 + 2 * size_t(N) + size_t(N) * N;
    std::vector<int32_t> h(nIn + nOut, 0);
    memcpy(h.data(), node_gpus, N * 4); memcpy(h.data() + N, node_compute, N * 4); memcpy(h.data() + 2 * N, node_mem_mb, N * 4);
    memcpy(h.data() + 3 * N, node_intra_bw, N * 4); memcpy(h.data() + 4 * N, inter_bw, size_t(N) * N * 4);
    int32_t* d = nullptr;
    TG_CUDA(poolAlloc(reinterpret_cast<void**>(&d), h.size() * 4, 0));
    cudaError_t e = cudaMemcpyAsync(d, h.data(), nIn * 4, cudaMemcpyHostToDevice, 0);
    if (e == cudaSuccess) {
        TgIslandsArgs A;
        A.N = N; A.gpus = d; A.comp = d + N; A.mem = d + 2 * N; A.intra = d + 3 * N; A.inter = d + 4 * N;
        A.epsC = eps_c; A.epsM = eps_m; A.epsI = eps_i;
        A.islandOf = d + nIn; A.K = A.islandOf + N; A.islandGpus = A.K + 1; A.islandCap = A.islandGpus + N; A.bw = A.islandCap + N;
        tgIslandsKernel<<<1, TG_ISL_NT>>>(A);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(h.data() + nIn, d + nIn, nOut * 4, cudaMemcpyDeviceToHost);
    cudaFreeAsync(d, 0);
    if (e != cudaSuccess) return fail(TG_ERR_CUDA, std::string("tg_islands_build: ") + cudaGetErrorString(e));
    const int32_t* o = h.data() + nIn;
    const int K = o[N];
    memcpy(island_of_node, o, N * 4);
    *k_out = K;
    memcpy(island_gpus, o + N + 1, K * 4);
    memcpy(island_cap_mb, o + 2 * N + 1, K * 4);
    memcpy(bw_gbps, o + 3 * N + 1, size_t(K) * K * 4);
    return TG_OK;
}

tg_status tg_release_cached_memory(void) {
    int dev = 0;
    TG_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_mu);
    if (dev >= 0 && dev < 64 && g_dev[dev].ready && g_dev[dev].pool) {
        TG_CUDA(cudaDeviceSynchronize());
        TG_CUDA(cudaMemPoolTrimTo(g_dev[dev].pool, 0));
    }
    return TG_OK;
}

tg_status tg_last_solver_kernel_ms(float* ms_out) {
    if (!ms_out) return fail(TG_ERR_NULL, "ms_out is NULL");
    if (!g_evA) return fail(TG_ERR_CUDA, "no solver kernel was launched on this thread");
    TG_CUDA(cudaEventSynchronize(g_evB));
    TG_CUDA(cudaEventElapsedTime(ms_out, g_evA, g_evB));
    return TG_OK;
}

tg_status tg_last_loader_kernel_ms(float* ms_out) {
    if (!ms_out) return fail(TG_ERR_NULL, "ms_out is NULL");
    if (!g_evL0) return fail(TG_ERR_CUDA, "no loader kernel was launched on this thread");
    TG_CUDA(cudaEventSynchronize(g_evL1));
    TG_CUDA(cudaEventElapsedTime(ms_out, g_evL0, g_evL1));
    return TG_OK;
}

tg_status tg_instance_read_time(tg_instance* inst, int32_t* time_out) {
    if (!inst || !time_out) return fail(TG_ERR_NULL, "NULL argument");
    TG_CUDA(cudaMemcpy(time_out, inst->time_us, size_t(inst->NS) * inst->K * inst->P * 4, cudaMemcpyDeviceToHost));
    return TG_OK;
}

}  // extern "C"
