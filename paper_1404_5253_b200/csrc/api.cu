// api.cu -- the C-ABI of libwpcd (include/wpcd.h): handles, host preparation (paper step 1,
// PAPER.md:310), argument checks and kernel launches.  No torch types, no CPU fallback.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <set>
#include <tuple>

#include "wigner_host.h"
#include "wpcd_internal.h"

namespace wpcd_detail {

static thread_local std::string t_error;
std::atomic<int64_t> g_launches{0};
DebugSwitches g_debug;

void set_error(const std::string& msg) { t_error = msg; }

cudaError_t raise_dyn_smem(const void* kernel, size_t bytes)
{
    static std::mutex mu;
    static std::map<std::pair<const void*, int>, size_t> have;      // (kernel, device) -> limit in force
    if (bytes <= 32 * 1024) return cudaSuccess;     // the default limit (48 KB, static shared memory included) covers it with room to spare
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    std::lock_guard<std::mutex> lock(mu);
    size_t& h = have[{kernel, dev}];
    if (bytes > h) {
        err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (err != cudaSuccess) return err;
        h = bytes;
    }
    return cudaSuccess;
}

static wpcd_status fail(wpcd_status code, const std::string& msg)
{
    set_error(msg);
    return code;
}

static wpcd_status cuda_fail(cudaError_t err, const char* where)
{
    return fail(WPCD_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(err));
}

static std::atomic<bool> g_trace_on{false};
struct TraceRec { int stage; cudaEvent_t e0, e1; };
static std::vector<TraceRec> g_trace;
static std::mutex g_trace_mutex;       // guards g_trace and g_trace_spare

static std::vector<cudaEvent_t> g_trace_spare;      // timing events are reused: creating one costs more than recording it

static cudaEvent_t trace_event()
{
    cudaEvent_t e = nullptr;
    std::lock_guard<std::mutex> lock(g_trace_mutex);
    if (!g_trace_spare.empty()) { e = g_trace_spare.back(); g_trace_spare.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}

StageTimer::StageTimer(int stage_, cudaStream_t st_) : stage(stage_), st(st_)
{
    if (!g_trace_on) return;
    e0 = trace_event(); e1 = trace_event();
    cudaEventRecord(e0, st);
}
StageTimer::~StageTimer()
{
    if (!e0) return;
    cudaEventRecord(e1, st);
    std::lock_guard<std::mutex> lock(g_trace_mutex);
    g_trace.push_back({stage, e0, e1});
}

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// ---- buffer cache (see wpcd_internal.h)
struct PoolEntry { void* ptr; size_t bytes; bool pinned; int device; };
static std::mutex g_pool_mutex;
static std::vector<PoolEntry> g_pool_free;
static std::map<void*, PoolEntry> g_pool_live;
static const size_t POOL_MAX_ENTRIES = 64;
static const size_t POOL_MAX_BYTES = (size_t)1 << 30;

static void pool_release(const PoolEntry& e)
{
    if (e.pinned) cudaFreeHost(e.ptr); else cudaFree(e.ptr);
}

void* pool_alloc(size_t bytes, bool pinned, cudaError_t* err)
{
    bytes = align256(std::max<size_t>(bytes, 1));
    int dev = 0;
    cudaGetDevice(&dev);
    *err = cudaSuccess;
    {
        std::lock_guard<std::mutex> lock(g_pool_mutex);
        size_t best = g_pool_free.size();
        for (size_t k = 0; k < g_pool_free.size(); ++k) {
            const PoolEntry& e = g_pool_free[k];
            if (e.pinned != pinned || e.device != dev || e.bytes < bytes || e.bytes > 2 * bytes + 4096) continue;
            if (best == g_pool_free.size() || e.bytes < g_pool_free[best].bytes) best = k;
        }
        if (best != g_pool_free.size()) {
            PoolEntry e = g_pool_free[best];
            g_pool_free.erase(g_pool_free.begin() + best);
            g_pool_live[e.ptr] = e;
            return e.ptr;
        }
    }
    void* ptr = nullptr;
    *err = pinned ? cudaMallocHost(&ptr, bytes) : cudaMalloc(&ptr, bytes);
    if (*err != cudaSuccess) return nullptr;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    g_pool_live[ptr] = {ptr, bytes, pinned, dev};
    return ptr;
}

void pool_free(void* ptr)
{
    if (!ptr) return;
    std::vector<PoolEntry> drop;
    {
        std::lock_guard<std::mutex> lock(g_pool_mutex);
        auto it = g_pool_live.find(ptr);
        if (it == g_pool_live.end()) return;
        g_pool_free.push_back(it->second);
        g_pool_live.erase(it);
        size_t total = 0;
        for (auto& e : g_pool_free) total += e.bytes;
        while (!g_pool_free.empty() && (g_pool_free.size() > POOL_MAX_ENTRIES || total > POOL_MAX_BYTES)) {
            total -= g_pool_free.front().bytes;
            drop.push_back(g_pool_free.front());
            g_pool_free.erase(g_pool_free.begin());
        }
    }
    for (auto& e : drop) pool_release(e);
}

Workspace carve_workspace(const wpcd_channels* ch, int64_t nnz_geo, void* base)
{
    Workspace ws{};
    size_t off = 0;
    char* b = static_cast<char*>(base);
    auto take = [&](size_t bytes) { char* ptr = b ? b + off : nullptr; off += align256(bytes); return ptr; };
    ws.geo_col = reinterpret_cast<int32_t*>(take(sizeof(int32_t) * (size_t)nnz_geo));
    ws.geo_row = reinterpret_cast<int32_t*>(take(sizeof(int32_t) * (size_t)nnz_geo));
    ws.geo_phi = reinterpret_cast<double2*>(take(sizeof(double2) * (size_t)nnz_geo));
    ws.chunk = 0;
    ws.moments = nullptr;
    ws.elem_rec = nullptr;
    ws.counters = nullptr;
    ws.n_chunks = 0;
    if (ch && !ch->swave_single) {
        ws.elem_rec = reinterpret_cast<int4*>(take(sizeof(int4) * (size_t)nnz_geo));
        // moment block: at most ~64 MiB (it stays in L2 between the kernel that writes it and the one that reads it), a
        // multiple of 32 elements
        int64_t chunk = (int64_t)((64ull << 20) / (sizeof(double) * (size_t)std::max(ch->n_mu, 1)));
        chunk = std::max<int64_t>(32, (chunk / 32) * 32);
        chunk = std::min<int64_t>(chunk, ((nnz_geo + 31) / 32) * 32);
        chunk = std::max<int64_t>(chunk, 32);
        ws.chunk = chunk;
        ws.n_chunks = (nnz_geo + chunk - 1) / chunk;
        ws.counters = reinterpret_cast<unsigned int*>(take(sizeof(unsigned int) * (size_t)std::max<int64_t>(ws.n_chunks, 1)));
        ws.moments = reinterpret_cast<double*>(take(sizeof(double) * (size_t)chunk * (size_t)ch->n_mu));
    }
    ws.bytes = off;
    return ws;
}

static void free_channels_device(wpcd_channels* c)
{
    if (c->ncoupled_dev) cudaDeviceSynchronize();   // the tables go back to the buffer cache: no kernel may still read them
    pool_free(c->tables_dev);
    c->tables_dev = nullptr;
}

template <class T>
static cudaError_t upload(T** dst, const std::vector<T>& src)
{
    size_t bytes = sizeof(T) * std::max<size_t>(src.size(), 1);
    cudaError_t err = cudaSuccess;
    *dst = static_cast<T*>(pool_alloc(bytes, false, &err));
    if (err != cudaSuccess) return err;
    if (!src.empty()) err = cudaMemcpy(*dst, src.data(), sizeof(T) * src.size(), cudaMemcpyHostToDevice);
    return err;
}

// Finish a channel handle whose host table (channel_l, pairs, terms) is filled in.
static wpcd_status finalize_channels(wpcd_channels* c)
{
    c->n_terms = (int64_t)c->term_g.size();
    // checks
    for (int a = 0; a < c->n_ch; ++a)
        if (c->channel_l[a] < 0 || c->channel_l[a] > WPCD_MAX_L) return fail(WPCD_ERR_UNSUPPORTED, "channel l beyond WPCD_MAX_L");
    for (int pidx = 0; pidx < c->n_pairs; ++pidx) {
        int ga = c->pair_gamma[pidx], gb = c->pair_gammap[pidx];
        if (ga < 0 || ga >= c->n_ch || gb < 0 || gb >= c->n_ch) return fail(WPCD_ERR_INVALID_ARG, "pair channel index out of range");
        if (pidx > 0 && std::make_pair(c->pair_gamma[pidx - 1], c->pair_gammap[pidx - 1]) >= std::make_pair(ga, gb))
            return fail(WPCD_ERR_INVALID_ARG, "pairs must be sorted ascending by (gamma, gamma') without repeats");
        if (c->term_ptr[pidx + 1] < c->term_ptr[pidx]) return fail(WPCD_ERR_INVALID_ARG, "term_ptr not monotone");
        if (c->term_ptr[pidx + 1] == c->term_ptr[pidx]) return fail(WPCD_ERR_INVALID_ARG, "a listed channel pair has no terms (leave uncoupled pairs out)");
    }
    // ---- merged coefficients per pair, monomial (A, k) = (l1 + l1', k)
    c->k_max = 0; c->l_max = 0; c->n_coef = 0;
    typedef std::pair<int, int> Mono;                           // (A, k)
    std::vector<std::map<Mono, double>> pair_coef(c->n_pairs);
    std::map<std::pair<int, int>, std::set<Mono>> ll_mono;      // (l, l') -> monomials used by any pair
    for (int pidx = 0; pidx < c->n_pairs; ++pidx) {
        int l = c->channel_l[c->pair_gamma[pidx]], lp = c->channel_l[c->pair_gammap[pidx]];
        c->l_max = std::max(c->l_max, std::max(l, lp));
        for (int64_t t = c->term_ptr[pidx]; t < c->term_ptr[pidx + 1]; ++t) {
            int k = c->term_k[t], l1 = c->term_l1[t], l1p = c->term_l1p[t];
            if (k < 0 || k > WPCD_MAX_K) return fail(WPCD_ERR_UNSUPPORTED, "Legendre order k beyond WPCD_MAX_K");
            if (l1 < 0 || l1 > l || l1p < 0 || l1p > lp) return fail(WPCD_ERR_INVALID_ARG, "l1 / l1' out of range");
            c->k_max = std::max(c->k_max, k);
            pair_coef[pidx][Mono(l1 + l1p, k)] += c->term_g[t];
        }
        for (auto& kv : pair_coef[pidx]) ll_mono[std::make_pair(l, lp)].insert(kv.first);
        c->n_coef += (int64_t)pair_coef[pidx].size();
    }
    // coupling structure
    c->ncoupled.assign(c->n_ch, 0);
    std::vector<int32_t> pair_ci(c->n_pairs);
    for (int pidx = 0; pidx < c->n_pairs; ++pidx) pair_ci[pidx] = c->ncoupled[c->pair_gamma[pidx]]++;
    std::vector<int64_t> chan_off(c->n_ch + 1, 0);
    for (int a = 0; a < c->n_ch; ++a) chan_off[a + 1] = chan_off[a] + c->ncoupled[a];
    c->total_coupled = chan_off[c->n_ch];
    c->coupled_gp.assign(c->n_pairs, 0);      // gamma' of block t of channel gamma, at chan_off[gamma] + t
    for (int pidx = 0; pidx < c->n_pairs; ++pidx) c->coupled_gp[chan_off[c->pair_gamma[pidx]] + pair_ci[pidx]] = c->pair_gammap[pidx];
    c->run_ptr.assign(1, 0); c->runs.clear(); c->first_gamma = -1;
    for (int a = 0; a < c->n_ch; ++a) {
        for (int t = 0; t < c->ncoupled[a];) {
            const int g0 = c->coupled_gp[chan_off[a] + t];
            int len = 1;
            while (t + len < c->ncoupled[a] && c->coupled_gp[chan_off[a] + t + len] == g0 + len) ++len;
            c->runs.push_back(make_int4(t, g0, len, 0));
            t += len;
        }
        c->run_ptr.push_back((int32_t)c->runs.size());
        if (c->first_gamma < 0 && c->ncoupled[a] > 0) { c->first_gamma = a; c->first_gp = c->coupled_gp[chan_off[a]]; }
    }
    // ---- moment row: one block per (l, l') with its distinct monomials; (l,l') list; (k,l,l') triples
    std::map<std::pair<int, int>, int> ll_index;
    c->ll_pack.clear();
    for (auto& kv : ll_mono) { ll_index[kv.first] = (int)c->ll_pack.size(); c->ll_pack.push_back(kv.first.first | (kv.first.second << 8)); }
    c->n_ll = (int)c->ll_pack.size();
    std::map<std::pair<int, int>, int> trip_index;   // (ll, k), sorted by (ll, k)
    for (auto& kv : ll_mono)
        for (auto& ak : kv.second) trip_index.emplace(std::make_pair(ll_index[kv.first], ak.second), 0);
    c->trip_pack.clear();
    for (auto& kv : trip_index) { kv.second = (int)c->trip_pack.size(); c->trip_pack.push_back(kv.first.second | (kv.first.first << 8)); }
    c->n_trip = (int)c->trip_pack.size();
    if (c->n_trip >= 65536) return fail(WPCD_ERR_UNSUPPORTED, "too many (k,l,l') combinations");
    std::map<std::tuple<int, int, int, int>, int> mu_index;   // (l, l', A, k) -> position in the moment row
    c->mu_pack.clear(); c->ab_pack.clear();
    std::map<std::pair<int, int>, int> ab_index;
    for (auto& kv : ll_mono) {
        int l = kv.first.first, lp = kv.first.second, ll = ll_index[kv.first];
        for (auto& ak : kv.second) {
            int A = ak.first, k = ak.second, B = l + lp - A;
            auto ab = ab_index.emplace(std::make_pair(A + 1, B + 1), (int)c->ab_pack.size());
            if (ab.second) c->ab_pack.push_back((A + 1) | ((B + 1) << 8));
            mu_index[std::make_tuple(l, lp, A, k)] = (int)c->mu_pack.size();
            c->mu_pack.push_back(trip_index[std::make_pair(ll, k)] | (ab.first->second << 16));
        }
    }
    c->n_ab = (int)c->ab_pack.size();
    if (c->n_ab >= 32768) return fail(WPCD_ERR_UNSUPPORTED, "too many cos/sin exponent pairs");
    c->n_mu = (int)c->mu_pack.size();
    // the same per monomial with the triple resolved: offset k IS + (l,l') into the I table of moments2_kernel (row stride
    // IS = 8 ceil(n_ll / 8) + 2) | exponent-pair index << 16 -- one table look-up per monomial instead of two dependent ones
    {
        const int IS = 8 * (((int)c->ll_pack.size() + 7) / 8) + 2;
        c->mu_ib_pack.resize(c->mu_pack.size());
        for (size_t m = 0; m < c->mu_pack.size(); ++m) {
            const int v = c->mu_pack[m], tp = c->trip_pack[v & 0xffff];
            const int o = (tp & 0xff) * IS + (tp >> 8);
            c->mu_ib_pack[m] = (o < 65536 ? o : 65535) | (v & ~0xffff);       // beyond 16 bits: moments2_kernel is not taken (K1 IS < 65536)
        }
    }
    // ---- contraction tables: (l, l') groups -> items (at most 8 pairs of the group with exactly the same monomials: for the nd
    // tables a class separates the (lambda, lambda') values, whose k-ranges differ);
    // every group's tables are one blob [items | pairs | idx | g] that the kernel copies to shared memory verbatim
    c->ct_groups.clear(); c->ct_blob.clear();
    c->ct_nmono_max = 0; c->ct_blob_max = 0; c->ct_ncoup_max = 0;
    for (int a = 0; a < c->n_ch; ++a) c->ct_ncoup_max = std::max(c->ct_ncoup_max, c->ncoupled[a]);
    for (auto& llkv : ll_mono) {       // the monomials of one (l, l') are one contiguous range of the moment row (mu_index is ordered by (l, l'))
        const int l = llkv.first.first, lp = llkv.first.second;
        int mu_lo = INT32_MAX, mu_hi = -1;
        for (auto& ak : llkv.second) {
            const int mu = mu_index[std::make_tuple(l, lp, ak.first, ak.second)];
            mu_lo = std::min(mu_lo, mu); mu_hi = std::max(mu_hi, mu);
        }
        // the group's pairs sorted into classes: exactly the same monomials
        std::map<std::vector<Mono>, std::vector<int>> classes;
        for (int pidx = 0; pidx < c->n_pairs; ++pidx) {
            if (c->channel_l[c->pair_gamma[pidx]] != l || c->channel_l[c->pair_gammap[pidx]] != lp) continue;
            std::vector<Mono> sig;
            for (auto& kv : pair_coef[pidx]) sig.push_back(kv.first);
            classes[sig].push_back(pidx);
        }
        std::vector<wpcd_ct_item> items;
        std::vector<int4> prs;              // per pair: (prefix of ncoupled over gamma, ncoupled(gamma), rank of gamma' in the row, gamma')
        std::vector<int32_t> idx;
        std::vector<double> gfr;
        auto pad16 = [](size_t b) { return (b + 15) & ~(size_t)15; };
        auto blob_size = [&](size_t ni, size_t npr, size_t nidx, size_t ng) {
            return pad16(sizeof(wpcd_ct_item) * ni) + pad16(sizeof(int4) * npr) + pad16(sizeof(int32_t) * nidx) + pad16(sizeof(double) * ng);
        };
        auto flush = [&]() {             // the items gathered so far become one group
            if (items.empty()) return;
            wpcd_ct_group g;
            g.mu_lo = mu_lo; g.n_mono = mu_hi - mu_lo + 1; g.n_items = (int32_t)items.size();
            g.blob_off = (int32_t)c->ct_blob.size();
            g.pairs_off = (int32_t)pad16(sizeof(wpcd_ct_item) * items.size());
            g.idx_off = g.pairs_off + (int32_t)pad16(sizeof(int4) * prs.size());
            g.g_off = g.idx_off + (int32_t)pad16(sizeof(int32_t) * idx.size());
            g.blob_bytes = g.g_off + (int32_t)pad16(sizeof(double) * gfr.size());
            c->ct_blob.resize(c->ct_blob.size() + g.blob_bytes, 0);
            unsigned char* base = c->ct_blob.data() + g.blob_off;
            std::memcpy(base, items.data(), sizeof(wpcd_ct_item) * items.size());
            std::memcpy(base + g.pairs_off, prs.data(), sizeof(int4) * prs.size());
            std::memcpy(base + g.idx_off, idx.data(), sizeof(int32_t) * idx.size());
            std::memcpy(base + g.g_off, gfr.data(), sizeof(double) * gfr.size());
            c->ct_nmono_max = std::max(c->ct_nmono_max, g.n_mono);
            c->ct_blob_max = std::max(c->ct_blob_max, g.blob_bytes);
            c->ct_groups.push_back(g);
            items.clear(); prs.clear(); idx.clear(); gfr.clear();
        };
        for (auto& kv : classes) {
            const std::vector<Mono>& sig = kv.first;
            const int ns = (int)sig.size(), kt = (ns + 3) / 4;
            for (size_t p_first = 0; p_first < kv.second.size(); p_first += 8) {
                const int np = (int)std::min<size_t>(8, kv.second.size() - p_first);
                // a group's blob stays below WPCD_CT_BLOB_BYTES (an (l, l') with many pairs becomes several groups)
                if (blob_size(items.size() + 1, prs.size() + np, idx.size() + 4 * kt, gfr.size() + (size_t)kt * np * 4) > WPCD_CT_BLOB_BYTES) flush();
                items.push_back({np, kt, (int32_t)idx.size(), (int32_t)gfr.size(), (int32_t)prs.size(), 0, 0, 0});
                for (int q = 0; q < np; ++q) {
                    const int pidx = kv.second[p_first + q], ga = c->pair_gamma[pidx];
                    prs.push_back(make_int4((int)chan_off[ga], c->ncoupled[ga], pair_ci[pidx], c->pair_gammap[pidx]));
                }
                for (int m = 0; m < 4 * kt; ++m) {
                    const Mono& mo = sig[std::min(m, ns - 1)];
                    idx.push_back(mu_index[std::make_tuple(l, lp, mo.first, mo.second)] - mu_lo);
                }
                for (int k = 0; k < kt; ++k)            // [k][pair][4]: only the item's own pairs are stored
                    for (int q = 0; q < np; ++q)
                        for (int mm = 0; mm < 4; ++mm) {
                            const int m = 4 * k + mm;
                            gfr.push_back(m < ns ? pair_coef[kv.second[p_first + q]][sig[m]] : 0.0);
                        }
            }
        }
        flush();
    }
    c->swave_single = (c->n_ch == 1 && c->n_pairs == 1 && c->n_terms == 1 && c->channel_l[0] == 0 && c->term_k[0] == 0);
    if (c->swave_single) c->g0 = c->term_g[0];
    // device tables (skipped when the process has no CUDA device: the host-side table stays
    // inspectable, every compute call then fails with WPCD_ERR_CUDA)
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) { cudaGetLastError(); return WPCD_OK; }
    // all device tables in ONE allocation and ONE copy (eight separate synchronous copies cost ~55 us per handle)
    auto pad = [](size_t b) { return (b + 255) & ~(size_t)255; };
    constexpr int NT = 12;
    const size_t sz[NT] = {sizeof(int32_t) * c->ncoupled.size(), sizeof(int64_t) * chan_off.size(), sizeof(int32_t) * c->coupled_gp.size(),
                           sizeof(int32_t) * c->ll_pack.size(),  sizeof(int32_t) * c->trip_pack.size(), sizeof(int32_t) * c->mu_pack.size(),
                           sizeof(int32_t) * c->ab_pack.size(),  sizeof(wpcd_ct_group) * c->ct_groups.size(), c->ct_blob.size(),
                           sizeof(int32_t) * c->run_ptr.size(),  sizeof(int4) * c->runs.size(), sizeof(int32_t) * c->mu_ib_pack.size()};
    const void* src[NT] = {c->ncoupled.data(), chan_off.data(), c->coupled_gp.data(), c->ll_pack.data(), c->trip_pack.data(),
                           c->mu_pack.data(), c->ab_pack.data(), c->ct_groups.data(), c->ct_blob.data(), c->run_ptr.data(),
                           c->runs.data(), c->mu_ib_pack.data()};
    size_t off[NT + 1];
    off[0] = 0;
    for (int k = 0; k < NT; ++k) off[k + 1] = off[k] + pad(std::max<size_t>(sz[k], 1));
    std::vector<unsigned char> blob(off[NT], 0);
    for (int k = 0; k < NT; ++k)
        if (sz[k]) std::memcpy(blob.data() + off[k], src[k], sz[k]);
    cudaError_t err = cudaSuccess;
    c->tables_dev = static_cast<unsigned char*>(pool_alloc(off[NT], false, &err));
    if (err == cudaSuccess) err = cudaMemcpy(c->tables_dev, blob.data(), off[NT], cudaMemcpyHostToDevice);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_channels_create");
    c->ncoupled_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[0]);
    c->chan_off_dev = reinterpret_cast<int64_t*>(c->tables_dev + off[1]);
    c->coupled_gp_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[2]);
    c->ll_pack_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[3]);
    c->trip_pack_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[4]);
    c->mu_pack_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[5]);
    c->ab_pack_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[6]);
    c->ct_groups_dev = reinterpret_cast<wpcd_ct_group*>(c->tables_dev + off[7]);
    c->ct_blob_dev = c->tables_dev + off[8];
    c->run_ptr_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[9]);
    c->runs_dev = reinterpret_cast<int4*>(c->tables_dev + off[10]);
    c->mu_ib_pack_dev = reinterpret_cast<int32_t*>(c->tables_dev + off[11]);
    return WPCD_OK;
}

}  // namespace wpcd_detail

using namespace wpcd_detail;

extern "C" {

const char* wpcd_last_error(void) { return t_error.c_str(); }

wpcd_status wpcd_grid_create(const double* p_nodes, int n_p, const double* q_nodes, int n_q, wpcd_grid** out)
{
    if (!p_nodes || !q_nodes || !out) return fail(WPCD_ERR_INVALID_ARG, "wpcd_grid_create: null pointer");
    *out = nullptr;
    if (n_p < 1 || n_q < 1) return fail(WPCD_ERR_INVALID_ARG, "wpcd_grid_create: n_p, n_q must be >= 1");
    if ((int64_t)n_p * n_q > (int64_t)INT32_MAX / 2) return fail(WPCD_ERR_OVERFLOW, "wpcd_grid_create: n_p*n_q too large");
    for (int i = 0; i <= n_p; ++i)
        if (!std::isfinite(p_nodes[i]) || (i == 0 ? p_nodes[0] < 0.0 : !(p_nodes[i] > p_nodes[i - 1])))
            return fail(WPCD_ERR_NOT_MONOTONE, "wpcd_grid_create: p nodes must be finite, >= 0 and strictly increasing");
    for (int i = 0; i <= n_q; ++i)
        if (!std::isfinite(q_nodes[i]) || (i == 0 ? q_nodes[0] < 0.0 : !(q_nodes[i] > q_nodes[i - 1])))
            return fail(WPCD_ERR_NOT_MONOTONE, "wpcd_grid_create: q nodes must be finite, >= 0 and strictly increasing");
    wpcd_grid* g = new (std::nothrow) wpcd_grid();
    if (!g) return fail(WPCD_ERR_ALLOC, "wpcd_grid_create: out of host memory");
    g->n_p = n_p; g->n_q = n_q;
    g->p.assign(p_nodes, p_nodes + n_p + 1);
    g->q.assign(q_nodes, q_nodes + n_q + 1);
    // one device block: p | q | ctrl | stage_off | stage_len (256-byte aligned pieces); one pinned block
    const size_t n_geo = (size_t)n_p * n_q;
    const size_t o_q = align256(sizeof(double) * (n_p + 1)), o_ctrl = o_q + align256(sizeof(double) * (n_q + 1));
    const size_t o_off = o_ctrl + 256, o_len = o_off + align256(sizeof(int32_t) * n_geo);
    const size_t total = o_len + align256(sizeof(int32_t) * n_geo);
    cudaError_t err = cudaSuccess;
    g->block_dev = static_cast<char*>(pool_alloc(total, false, &err));
    if (err == cudaSuccess) g->ctrl_pinned = static_cast<int32_t*>(pool_alloc(256, true, &err));
    if (err == cudaSuccess) {
        g->p_dev = reinterpret_cast<double*>(g->block_dev);
        g->q_dev = reinterpret_cast<double*>(g->block_dev + o_q);
        g->ctrl = reinterpret_cast<int32_t*>(g->block_dev + o_ctrl);
        g->stage_off = reinterpret_cast<int32_t*>(g->block_dev + o_off);
        g->stage_len = reinterpret_cast<int32_t*>(g->block_dev + o_len);
        // p | q | zeroed control words go up in ONE copy (three synchronous operations cost ~20 us per handle)
        std::vector<unsigned char> head(o_off, 0);
        std::memcpy(head.data(), p_nodes, sizeof(double) * (n_p + 1));
        std::memcpy(head.data() + o_q, q_nodes, sizeof(double) * (n_q + 1));
        err = cudaMemcpy(g->block_dev, head.data(), o_off, cudaMemcpyHostToDevice);
    }
    if (err != cudaSuccess) { wpcd_grid_destroy(g); return cuda_fail(err, "wpcd_grid_create"); }
    *out = g;
    return WPCD_OK;
}

void wpcd_grid_destroy(wpcd_grid* g)
{
    if (!g) return;
    if (g->select_ready) cudaDeviceSynchronize();   // scratch goes back to the cache: no kernel may still use it
    pool_free(g->block_dev); pool_free(g->stage_col); pool_free(g->stage_ext); pool_free(g->ctrl_pinned);
    if (g->count_event) cudaEventDestroy(g->count_event);
    if (g->rowptr_event) cudaEventDestroy(g->rowptr_event);
    delete g;
}

wpcd_status wpcd_channels_create(int model, int two_J, int parity, int two_T, int j_pair_max, double g0, wpcd_channels** out)
{
    if (!out) return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_create: null pointer");
    *out = nullptr;
    wpcd_channels* c = new (std::nothrow) wpcd_channels();
    if (!c) return fail(WPCD_ERR_ALLOC, "wpcd_channels_create: out of host memory");
    c->model = model;
    if (model == WPCD_SPINLESS_SWAVE) {
        if (!std::isfinite(g0)) { delete c; return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_create: g0 not finite"); }
        c->n_ch = 1; c->n_pairs = 1;
        c->qn.assign(6, 0); c->channel_l = {0};
        c->pair_gamma = {0}; c->pair_gammap = {0}; c->term_ptr = {0, 1};
        c->term_k = {0}; c->term_l1 = {0}; c->term_l1p = {0}; c->term_g = {g0};
    } else if (model == WPCD_ND) {
        if (two_J < 1 || (two_J & 1) == 0 || (parity != 1 && parity != -1) || two_T != 1 || j_pair_max < 0 || j_pair_max > 6) {
            delete c;
            return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_create: need odd two_J >= 1, parity = +-1, two_T = 1, 0 <= j_pair_max <= 6");
        }
        std::vector<wpcd_host::Channel> chs = wpcd_host::enumerate_channels(two_J, parity, j_pair_max);
        std::vector<wpcd_host::Pair> pairs = wpcd_host::g_table(chs, two_J, two_T);
        c->n_ch = (int)chs.size(); c->n_pairs = (int)pairs.size();
        for (auto& ch : chs) {
            c->channel_l.push_back(ch.l);
            int32_t v[6] = {ch.l, ch.s, ch.j, ch.t, ch.lam, ch.two_I};
            c->qn.insert(c->qn.end(), v, v + 6);
        }
        c->term_ptr.push_back(0);
        for (auto& pr : pairs) {
            c->pair_gamma.push_back(pr.gamma); c->pair_gammap.push_back(pr.gammap);
            for (auto& t : pr.terms) { c->term_k.push_back(t.k); c->term_l1.push_back(t.l1); c->term_l1p.push_back(t.l1p); c->term_g.push_back(t.g); }
            c->term_ptr.push_back((int64_t)c->term_g.size());
        }
    } else {
        delete c;
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_create: unknown model");
    }
    wpcd_status st = finalize_channels(c);
    if (st != WPCD_OK) { wpcd_channels_destroy(c); return st; }
    *out = c;
    return WPCD_OK;
}

wpcd_status wpcd_channels_create_from_table(int n_channels, const int32_t* channel_l, int n_pairs, const int32_t* pair_gamma,
                                            const int32_t* pair_gammap, const int64_t* term_ptr, const int32_t* term_k,
                                            const int32_t* term_l1, const int32_t* term_l1p, const double* term_g,
                                            wpcd_channels** out)
{
    if (!out) return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_create_from_table: null pointer");
    *out = nullptr;
    if (n_channels < 1 || n_pairs < 0 || !channel_l || !term_ptr || (n_pairs > 0 && (!pair_gamma || !pair_gammap)))
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_create_from_table: bad sizes or null pointer");
    int64_t n_terms = term_ptr[n_pairs];
    if (term_ptr[0] != 0 || n_terms < 0 || (n_terms > 0 && (!term_k || !term_l1 || !term_l1p || !term_g)))
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_create_from_table: bad term arrays");
    wpcd_channels* c = new (std::nothrow) wpcd_channels();
    if (!c) return fail(WPCD_ERR_ALLOC, "out of host memory");
    c->model = -1;
    c->n_ch = n_channels; c->n_pairs = n_pairs;
    c->channel_l.assign(channel_l, channel_l + n_channels);
    c->qn.assign((size_t)n_channels * 6, 0);
    for (int a = 0; a < n_channels; ++a) c->qn[(size_t)a * 6] = channel_l[a];
    c->pair_gamma.assign(pair_gamma, pair_gamma + n_pairs);
    c->pair_gammap.assign(pair_gammap, pair_gammap + n_pairs);
    c->term_ptr.assign(term_ptr, term_ptr + n_pairs + 1);
    c->term_k.assign(term_k, term_k + n_terms);
    c->term_l1.assign(term_l1, term_l1 + n_terms);
    c->term_l1p.assign(term_l1p, term_l1p + n_terms);
    c->term_g.assign(term_g, term_g + n_terms);
    wpcd_status st = finalize_channels(c);
    if (st != WPCD_OK) { wpcd_channels_destroy(c); return st; }
    *out = c;
    return WPCD_OK;
}

void wpcd_channels_destroy(wpcd_channels* c)
{
    if (!c) return;
    free_channels_device(c);
    delete c;
}

int wpcd_channels_count(const wpcd_channels* c) { return c ? c->n_ch : 0; }
int wpcd_channels_pairs(const wpcd_channels* c) { return c ? c->n_pairs : 0; }
int64_t wpcd_channels_terms(const wpcd_channels* c) { return c ? c->n_terms : 0; }
int wpcd_channels_monomials(const wpcd_channels* c) { return c ? c->n_mu : 0; }
int64_t wpcd_channels_coefficients(const wpcd_channels* c) { return c ? c->n_coef : 0; }

wpcd_status wpcd_channels_get_quantum_numbers(const wpcd_channels* c, int32_t* out)
{
    if (!c || !out) return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_get_quantum_numbers: null pointer");
    std::memcpy(out, c->qn.data(), sizeof(int32_t) * c->qn.size());
    return WPCD_OK;
}

wpcd_status wpcd_channels_get_table(const wpcd_channels* c, int32_t* pair_gamma, int32_t* pair_gammap, int64_t* term_ptr,
                                    int32_t* term_k, int32_t* term_l1, int32_t* term_l1p, double* term_g)
{
    if (!c || !pair_gamma || !pair_gammap || !term_ptr || !term_k || !term_l1 || !term_l1p || !term_g)
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_channels_get_table: null pointer");
    std::memcpy(pair_gamma, c->pair_gamma.data(), sizeof(int32_t) * c->n_pairs);
    std::memcpy(pair_gammap, c->pair_gammap.data(), sizeof(int32_t) * c->n_pairs);
    std::memcpy(term_ptr, c->term_ptr.data(), sizeof(int64_t) * (c->n_pairs + 1));
    std::memcpy(term_k, c->term_k.data(), sizeof(int32_t) * c->n_terms);
    std::memcpy(term_l1, c->term_l1.data(), sizeof(int32_t) * c->n_terms);
    std::memcpy(term_l1p, c->term_l1p.data(), sizeof(int32_t) * c->n_terms);
    std::memcpy(term_g, c->term_g.data(), sizeof(double) * c->n_terms);
    return WPCD_OK;
}

int64_t wpcd_rows(const wpcd_grid* g, const wpcd_channels* c) { return (g && c) ? (int64_t)c->n_ch * g->n_p * g->n_q : 0; }
int64_t wpcd_geo_rows(const wpcd_grid* g) { return g ? (int64_t)g->n_p * g->n_q : 0; }

// Selection pass on grid g: predicate, per-row counts, staged verdicts, scan, and (when c is
// given) the row pointer of the full matrix.  Synchronises the stream (the caller needs nnz_geo);
// repeats the pass with a larger staging area if it overflowed.
static wpcd_status run_selection(const wpcd_grid* g, const wpcd_channels* c, int32_t* geo_row_ptr_dev, int64_t* row_ptr_dev,
                                 cudaStream_t st, const char* who)
{
    const int n_geo = g->n_p * g->n_q;
    int64_t want = g->stage_cap > 0 ? g->stage_cap : std::max<int64_t>(1024, (int64_t)48 * n_geo);
    for (int attempt = 0; attempt < 3; ++attempt) {
        cudaError_t err = ensure_stage(g, want);
        if (err != cudaSuccess) return cuda_fail(err, who);
        g->stage_valid = false;
        // the host waits for the selection pass only (an event behind the read-back of its result); the expansion to the
        // full row pointer is queued behind it and runs while the call returns
        if (!g->count_event) {
            err = cudaEventCreateWithFlags(&g->count_event, cudaEventDisableTiming);
            if (err == cudaSuccess) err = cudaEventCreateWithFlags(&g->rowptr_event, cudaEventDisableTiming);
            if (err != cudaSuccess) return cuda_fail(err, who);
        }
        err = launch_geo_select(g, geo_row_ptr_dev, st);
        if (err == cudaSuccess) err = cudaMemcpyAsync(g->ctrl_pinned, g->ctrl + 4, sizeof(int32_t) * 4, cudaMemcpyDeviceToHost, st);
        if (err == cudaSuccess) err = cudaEventRecord(g->count_event, st);
        if (err == cudaSuccess && c) err = launch_rowptr(g, c, geo_row_ptr_dev, row_ptr_dev, st);
        if (err == cudaSuccess && c) err = cudaEventRecord(g->rowptr_event, st);     // for a build on another stream
        g->count_stream = st;
        if (err == cudaSuccess) err = cudaEventSynchronize(g->count_event);
        if (err != cudaSuccess) return cuda_fail(err, who);
        if (g->ctrl_pinned[1] == 0) {
            g->stage_valid = true;
            g->stage_nnz_geo = g->ctrl_pinned[2];
            return WPCD_OK;
        }
        if (g->ctrl_pinned[0] < 0) return fail(WPCD_ERR_OVERFLOW, std::string(who) + ": more than 2^31 candidate cell pairs");
        want = (int64_t)g->ctrl_pinned[0] + (int64_t)g->ctrl_pinned[0] / 8 + 1024;
    }
    return fail(WPCD_ERR_ALLOC, std::string(who) + ": staging area kept overflowing");
}

wpcd_status wpcd_perm_count(const wpcd_grid* g, const wpcd_channels* c, int n_quad, void* cuda_stream, int64_t* row_ptr_dev,
                            int32_t* geo_row_ptr_dev, int64_t* nnz_out, int64_t* nnz_geo_out)
{
    if (!g || !c || !row_ptr_dev || !geo_row_ptr_dev || !nnz_out || !nnz_geo_out)
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_count: null pointer");
    n_quad &= ~(WPCD_RULE_KINK_SPLIT | WPCD_RULE_ANALYTIC_U);       // the pattern does not depend on the rule
    if (n_quad < 1 || n_quad > WPCD_MAX_QUAD) return fail(WPCD_ERR_UNSUPPORTED, "wpcd_perm_count: n_quad out of range");
    if (!c->ncoupled_dev) return fail(WPCD_ERR_CUDA, "wpcd_perm_count: channel tables are not on a device (no CUDA device?)");
    int64_t rows = wpcd_rows(g, c);
    if (rows > (int64_t)INT32_MAX) return fail(WPCD_ERR_OVERFLOW, "wpcd_perm_count: column index would not fit int32");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    wpcd_status s = run_selection(g, c, geo_row_ptr_dev, row_ptr_dev, st, "wpcd_perm_count");
    if (s != WPCD_OK) return s;
    int64_t nnz_geo = g->stage_nnz_geo;
    *nnz_geo_out = nnz_geo;
    *nnz_out = nnz_geo * c->total_coupled;
    return WPCD_OK;
}

size_t wpcd_perm_workspace_bytes(const wpcd_channels* c, int64_t nnz_geo)
{
    if (!c || nnz_geo < 0) return 0;
    return carve_workspace(c, nnz_geo, nullptr).bytes;
}

wpcd_status wpcd_perm_build(const wpcd_grid* g, const wpcd_channels* c, int n_quad, void* cuda_stream, const int64_t* row_ptr_dev,
                            const int32_t* geo_row_ptr_dev, void* workspace_dev, size_t workspace_bytes, int32_t* col_idx_dev,
                            double* values_dev)
{
    if (!g || !c || !row_ptr_dev || !geo_row_ptr_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_build: null pointer");
    const bool analytic = (n_quad & WPCD_RULE_ANALYTIC_U) != 0;
    const bool split = (n_quad & WPCD_RULE_KINK_SPLIT) != 0 || analytic;
    n_quad &= ~(WPCD_RULE_KINK_SPLIT | WPCD_RULE_ANALYTIC_U);
    if (analytic && !c->swave_single)
        return fail(WPCD_ERR_UNSUPPORTED, "wpcd_perm_build: WPCD_RULE_ANALYTIC_U is for the s-wave term (k = l = l' = 0) only");
    if (n_quad < 1 || n_quad > WPCD_MAX_QUAD) return fail(WPCD_ERR_UNSUPPORTED, "wpcd_perm_build: n_quad out of range");
    if (!c->ncoupled_dev) return fail(WPCD_ERR_CUDA, "wpcd_perm_build: channel tables are not on a device (no CUDA device?)");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!g->stage_valid) {
        // no selection pass has run on this handle (geo_row_ptr came from elsewhere): redo it into
        // a scratch copy of the row pointer so that the caller's array stays untouched
        int32_t* tmp = nullptr;
        const int n_geo = g->n_p * g->n_q;
        cudaError_t err = cudaMalloc(reinterpret_cast<void**>(&tmp), sizeof(int32_t) * (n_geo + 1));
        if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_build(selection scratch)");
        wpcd_status s = run_selection(g, nullptr, tmp, nullptr, st, "wpcd_perm_build");
        cudaFree(tmp);
        if (s != WPCD_OK) return s;
    }
    const int64_t nnz_geo = g->stage_nnz_geo;
    if (nnz_geo == 0 || c->total_coupled == 0) return WPCD_OK;
    if (g->rowptr_event && st != g->count_stream) {      // the count's row-pointer expansion may still run on its own stream
        cudaError_t werr = cudaStreamWaitEvent(st, g->rowptr_event, 0);
        if (werr != cudaSuccess) return cuda_fail(werr, "wpcd_perm_build");
    }
    if (!workspace_dev || !col_idx_dev || !values_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_build: null output or workspace");
    if ((reinterpret_cast<uintptr_t>(workspace_dev) & 255) != 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_build: workspace must be 256-byte aligned");
    Workspace ws = carve_workspace(c, nnz_geo, workspace_dev);
    if (workspace_bytes < ws.bytes) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_build: workspace too small");
    cudaError_t err = launch_geo_gather(g, geo_row_ptr_dev, ws.geo_col, ws.geo_row, ws.geo_phi, st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_build(index)");
    // Gauss-Legendre nodes / weights: computed once per order (host, long double Newton), then reused
    static std::mutex gl_mutex;
    static std::map<int, std::vector<double>> gl_cache;
    QuadRule qr;
    {
        std::lock_guard<std::mutex> lock(gl_mutex);
        std::vector<double>& tab = gl_cache[n_quad];
        if (tab.empty()) {
            tab.resize(2 * n_quad);
            wpcd_host::gauss_legendre(n_quad, tab.data(), tab.data() + n_quad);
        }
        std::memset(&qr, 0, sizeof(qr));
        std::memcpy(qr.xi, tab.data(), sizeof(double) * n_quad);
        std::memcpy(qr.w, tab.data() + n_quad, sizeof(double) * n_quad);
        for (int k = 1; k < WPCD_MAX_K + 2; ++k) qr.invk[k] = 1.0 / k;
    }
    if (c->swave_single) err = launch_fill_swave(g, c, n_quad, analytic ? 2 : (split ? 1 : 0), qr, nnz_geo, ws, col_idx_dev, values_dev, st);
    else err = launch_fill_coupled(g, c, n_quad, split, qr, nnz_geo, ws, row_ptr_dev, geo_row_ptr_dev, col_idx_dev, values_dev, st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_build(fill)");
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                            const double* x_dev, double* y_dev, int n_vec, void* cuda_stream)
{
    if (rows < 0 || n_vec < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply: negative size");
    if (rows == 0 || n_vec == 0) return WPCD_OK;
    if (!row_ptr_dev || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply: null pointer");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t err = launch_spmv(rows, row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, n_vec, st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply");
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply_complex(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                    const double* x_dev, double* y_dev, int n_vec, void* cuda_stream)
{
    if (rows < 0 || n_vec < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_complex: negative size");
    if (rows == 0 || n_vec == 0) return WPCD_OK;
    if (!row_ptr_dev || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_complex: null pointer");
    if ((reinterpret_cast<uintptr_t>(x_dev) & 15) || (reinterpret_cast<uintptr_t>(y_dev) & 15))
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_complex: x and y must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t err = launch_spmv_interleaved(rows, row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, n_vec, 2, st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_complex");
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply_interleaved(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                        const double* x_dev, double* y_dev, int n_inter, void* cuda_stream)
{
    if (rows < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_interleaved: negative size");
    if (n_inter != 2 && n_inter != 4) return fail(WPCD_ERR_UNSUPPORTED, "wpcd_perm_apply_interleaved: n_inter must be 2 or 4");
    if (rows == 0) return WPCD_OK;
    if (!row_ptr_dev || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_interleaved: null pointer");
    if ((reinterpret_cast<uintptr_t>(x_dev) & 15) || (reinterpret_cast<uintptr_t>(y_dev) & 15))
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_interleaved: x and y must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t err = launch_spmv_interleaved(rows, row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, 1, n_inter, st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_interleaved");
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply_blocked(const wpcd_grid* g, const wpcd_channels* c, const int64_t* row_ptr_dev,
                                    const int32_t* geo_row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                    const double* x_dev, double* y_dev, int n_vec, void* cuda_stream)
{
    if (!g || !c) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked: null handle");
    if (n_vec < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked: negative size");
    const int64_t rows = wpcd_rows(g, c);
    if (rows == 0 || n_vec == 0) return WPCD_OK;
    if (!row_ptr_dev || !geo_row_ptr_dev || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked: null pointer");
    if (!c->ncoupled_dev) return fail(WPCD_ERR_CUDA, "wpcd_perm_apply_blocked: channel tables are not on a device (no CUDA device?)");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (c->total_coupled > 0 && (!col_idx_dev || !values_dev)) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked: null matrix arrays");
    cudaError_t err = launch_spmv_blocked(g, c, geo_row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, n_vec, st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_blocked");
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply_blocked_noalloc(const wpcd_grid* g, const wpcd_channels* c, const int64_t* row_ptr_dev,
                                            const int32_t* geo_row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                            const double* x_dev, double* y_dev, int n_vec, void* cuda_stream)
{
    if (!g || !c) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked_noalloc: null handle");
    if (n_vec < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked_noalloc: negative size");
    const int64_t rows = wpcd_rows(g, c);
    if (rows == 0 || n_vec == 0) return WPCD_OK;
    if (n_vec > 8) return fail(WPCD_ERR_UNSUPPORTED, "wpcd_perm_apply_blocked_noalloc: at most 8 vectors per call");
    if (rows > WPCD_NOALLOC_MAX_ROWS)
        return fail(WPCD_ERR_UNSUPPORTED, "wpcd_perm_apply_blocked_noalloc: " + std::to_string(rows) + " rows exceed WPCD_NOALLOC_MAX_ROWS = " +
                                              std::to_string(WPCD_NOALLOC_MAX_ROWS) + " (the fixed scratch array); use wpcd_perm_apply_blocked");
    if (c->n_ch > 64) return fail(WPCD_ERR_UNSUPPORTED, "wpcd_perm_apply_blocked_noalloc: more than 64 channels");
    if (!row_ptr_dev || !geo_row_ptr_dev || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked_noalloc: null pointer");
    if (!c->ncoupled_dev) return fail(WPCD_ERR_CUDA, "wpcd_perm_apply_blocked_noalloc: channel tables are not on a device (no CUDA device?)");
    if (c->total_coupled > 0 && (!col_idx_dev || !values_dev)) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked_noalloc: null matrix arrays");
    cudaError_t err = launch_spmv_blocked_noalloc(g, c, geo_row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, n_vec, static_cast<cudaStream_t>(cuda_stream));
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_blocked_noalloc");
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply_chain(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                  const double* x_dev, double* y_dev, int n_iter, void* cuda_stream)
{
    if (rows < 0 || n_iter < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_chain: negative size");
    if (rows == 0 || n_iter == 0) return WPCD_OK;
    if (!row_ptr_dev || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_chain: null pointer");
    if (x_dev + rows > y_dev && y_dev + (int64_t)n_iter * rows > x_dev)
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_chain: x overlaps y");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // the fused launch sizes its shared-memory slices from the number of nonzeros: one small read-back per call
    int64_t nnz = 0;
    cudaError_t nerr = cudaMemcpyAsync(&nnz, row_ptr_dev + rows, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    if (nerr == cudaSuccess) nerr = cudaStreamSynchronize(st);
    if (nerr != cudaSuccess) return cuda_fail(nerr, "wpcd_perm_apply_chain");
    if (nnz > 0 && (!col_idx_dev || !values_dev)) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_chain: null matrix arrays");
    int fused = 0;
    cudaError_t err = launch_spmv_chain(rows, row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, n_iter, nnz, st, &fused);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_chain");
    if (!fused) {
        const double* xin = x_dev;
        for (int k = 0; k < n_iter; ++k) {
            double* yk = y_dev + (int64_t)k * rows;
            err = launch_spmv(rows, row_ptr_dev, col_idx_dev, values_dev, xin, yk, 1, st);
            if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_chain");
            xin = yk;
        }
    }
    return WPCD_OK;
}

wpcd_status wpcd_block_apply(int n_channels, int n_p, int n_q, const double* a_dev, int transpose, const double* x_dev,
                             double* y_dev, int complex_vectors, void* cuda_stream)
{
    if (n_channels < 0 || n_p < 0 || n_q < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_block_apply: negative size");
    if (n_channels == 0 || n_p == 0 || n_q == 0) return WPCD_OK;
    if (!a_dev || !x_dev || !y_dev || x_dev == y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_block_apply: null pointer or x aliases y");
    cudaError_t err = launch_block_apply(n_channels, n_p, complex_vectors ? 2 * n_q : n_q, a_dev, transpose != 0, x_dev, y_dev,
                                         static_cast<cudaStream_t>(cuda_stream));
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_block_apply");
    return WPCD_OK;
}

wpcd_status wpcd_kernel_apply(int n_channels, int n_p, int n_q, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                              const double* values_dev, const double* o_dev, const double* v_dev, const double* g1_dev,
                              const double* x_dev, double* y_dev, double* scratch_dev, void* cuda_stream)
{
    if (n_channels < 0 || n_p < 0 || n_q < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_kernel_apply: negative size");
    const int64_t rows = (int64_t)n_channels * n_p * n_q;
    if (rows == 0) return WPCD_OK;
    if (!row_ptr_dev || !o_dev || !v_dev || !g1_dev || !x_dev || !y_dev || !scratch_dev)
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_kernel_apply: null pointer");
    if ((reinterpret_cast<uintptr_t>(x_dev) | reinterpret_cast<uintptr_t>(y_dev) | reinterpret_cast<uintptr_t>(scratch_dev) |
         reinterpret_cast<uintptr_t>(g1_dev)) & 15)
        return fail(WPCD_ERR_INVALID_ARG, "wpcd_kernel_apply: complex arrays must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double* t1 = scratch_dev;                 // [rows] complex
    double* t2 = scratch_dev + 2 * rows;      // [rows] complex
    cudaError_t err = launch_diag_scale(rows, g1_dev, x_dev, t1, st);                                   // G1 .* x
    if (err == cudaSuccess) err = launch_block_apply(n_channels, n_p, 2 * n_q, v_dev, false, t1, t2, st);  // V1
    if (err == cudaSuccess) err = launch_block_apply(n_channels, n_p, 2 * n_q, o_dev, true, t2, t1, st);   // O^T
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_kernel_apply");
    wpcd_status s = wpcd_perm_apply_complex(rows, row_ptr_dev, col_idx_dev, values_dev, t1, t2, 1, cuda_stream);   // P0
    if (s != WPCD_OK) return s;
    err = launch_block_apply(n_channels, n_p, 2 * n_q, o_dev, false, t2, y_dev, st);                    // O
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_kernel_apply");
    return WPCD_OK;
}

wpcd_status wpcd_neumann_terms(int n_channels, int n_p, int n_q, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                               const double* values_dev, const double* o_dev, const double* v_dev, const double* g1_dev,
                               const double* b_dev, int64_t element, int n_terms, double* terms_host, double* scratch_dev,
                               void* cuda_stream)
{
    const int64_t rows = (int64_t)n_channels * n_p * n_q;
    if (n_terms < 1 || !terms_host || !b_dev || !scratch_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_neumann_terms: bad arguments");
    if (element < 0 || element >= rows) return fail(WPCD_ERR_INVALID_ARG, "wpcd_neumann_terms: element out of range");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // scratch: [0, 2 rows) complex for wpcd_kernel_apply, then two complex vectors, then the picked terms
    double* ka_scratch = scratch_dev;
    double* va = scratch_dev + 4 * rows;
    double* vb = va + 2 * rows;
    double* picked = vb + 2 * rows;          // [n_terms] complex
    cudaError_t err = cudaMemcpyAsync(va, b_dev, sizeof(double) * 2 * rows, cudaMemcpyDeviceToDevice, st);
    for (int n = 0; n < n_terms && err == cudaSuccess; ++n) {
        err = cudaMemcpyAsync(picked + 2 * n, va + 2 * element, sizeof(double) * 2, cudaMemcpyDeviceToDevice, st);   // a_n = (K^n b)[element]
        if (err != cudaSuccess || n + 1 == n_terms) break;
        wpcd_status s = wpcd_kernel_apply(n_channels, n_p, n_q, row_ptr_dev, col_idx_dev, values_dev, o_dev, v_dev, g1_dev, va, vb,
                                          ka_scratch, cuda_stream);
        if (s != WPCD_OK) return s;
        std::swap(va, vb);
    }
    if (err == cudaSuccess) err = cudaMemcpyAsync(terms_host, picked, sizeof(double) * 2 * n_terms, cudaMemcpyDeviceToHost, st);
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_neumann_terms");
    return WPCD_OK;
}

wpcd_status wpcd_pade_sum(const double* terms_host, int n_terms, double* sum_out)
{
    if (!terms_host || !sum_out || n_terms < 1) return fail(WPCD_ERR_INVALID_ARG, "wpcd_pade_sum: bad arguments");
    // Wynn's epsilon algorithm on the partial sums: eps_{k+1}^{(n)} = eps_{k-1}^{(n+1)} + 1 / (eps_k^{(n+1)} - eps_k^{(n)});
    // the even columns are the Pade approximants [n+k / k] of the series at lambda = 1
    typedef std::complex<double> cplx;
    std::vector<cplx> prev(n_terms + 1, cplx(0.0, 0.0)), cur(n_terms), nxt;
    cplx run(0.0, 0.0);
    for (int n = 0; n < n_terms; ++n) { run += cplx(terms_host[2 * n], terms_host[2 * n + 1]); cur[n] = run; }
    cplx best = cur.back();
    for (int k = 0; (int)cur.size() > 1; ++k) {
        nxt.assign(cur.size() - 1, cplx(0.0, 0.0));
        bool ok = true;
        for (size_t n = 0; n + 1 < cur.size(); ++n) {
            cplx d = cur[n + 1] - cur[n];
            if (std::abs(d) == 0.0) { ok = false; break; }      // converged exactly: keep the last even column
            nxt[n] = prev[n + 1] + cplx(1.0, 0.0) / d;
        }
        if (!ok) break;
        prev = cur; cur = nxt;
        if ((k & 1) == 1) best = cur.back();                   // cur is now an even column
    }
    sum_out[0] = best.real(); sum_out[1] = best.imag();
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply_host(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                 const double* x_host, double* y_host, int n_vec, double* x_dev, double* y_dev, void* cuda_stream)
{
    if (rows < 0 || n_vec < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_host: negative size");
    if (rows == 0 || n_vec == 0) return WPCD_OK;
    if (!x_host || !y_host || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_host: null pointer");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    constexpr int CHUNK = 8;       // right-hand sides per pipeline stage (two passes of 4)
    if (n_vec <= CHUNK) {
        size_t bytes = sizeof(double) * (size_t)rows * (size_t)n_vec;
        cudaError_t err = cudaMemcpyAsync(x_dev, x_host, bytes, cudaMemcpyHostToDevice, st);
        if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host(H2D)");
        wpcd_status s = wpcd_perm_apply(rows, row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, n_vec, cuda_stream);
        if (s != WPCD_OK) return s;
        err = cudaMemcpyAsync(y_host, y_dev, bytes, cudaMemcpyDeviceToHost, st);
        if (err == cudaSuccess) err = cudaStreamSynchronize(st);
        if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host(D2H)");
        return WPCD_OK;
    }
    // Many right-hand sides: three-stage pipeline over chunks of CHUNK vectors -- upload of chunk k+1 (copy stream "up"),
    // products of chunk k (the caller's stream) and download of chunk k-1 (copy stream "down") run together, so the call
    // costs about the larger of the two copy directions instead of upload + products + download.
    struct HostPipe { cudaStream_t up = nullptr, down = nullptr; std::vector<cudaEvent_t> ev; };
    static std::mutex pipe_mutex;
    static std::map<int, HostPipe> pipes;
    std::lock_guard<std::mutex> lock(pipe_mutex);      // the call is synchronous; one pipelined host apply at a time
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host");
    HostPipe& hp = pipes[dev];
    if (!hp.up) {
        err = cudaStreamCreateWithFlags(&hp.up, cudaStreamNonBlocking);
        if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&hp.down, cudaStreamNonBlocking);
        if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host(streams)");
    }
    const int n_chunk = (n_vec + CHUNK - 1) / CHUNK;
    while ((int)hp.ev.size() < 2 * n_chunk) {
        cudaEvent_t e;
        err = cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
        if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host(events)");
        hp.ev.push_back(e);
    }
    // The uploads start at once -- they do not wait for what the caller's stream still holds (typically the build of the
    // matrix), only the products do; the scratch vectors must therefore not be in use by earlier asynchronous work.
    for (int k = 0; k < n_chunk; ++k) {
        const int v0 = k * CHUNK, nv = std::min(CHUNK, n_vec - v0);
        const size_t off = (size_t)v0 * (size_t)rows, bytes = sizeof(double) * (size_t)rows * (size_t)nv;
        err = cudaMemcpyAsync(x_dev + off, x_host + off, bytes, cudaMemcpyHostToDevice, hp.up);
        if (err == cudaSuccess) err = cudaEventRecord(hp.ev[2 * k], hp.up);
        if (err == cudaSuccess) err = cudaStreamWaitEvent(st, hp.ev[2 * k], 0);
        if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host(H2D)");
        wpcd_status s = wpcd_perm_apply(rows, row_ptr_dev, col_idx_dev, values_dev, x_dev + off, y_dev + off, nv, cuda_stream);
        if (s != WPCD_OK) return s;
        err = cudaEventRecord(hp.ev[2 * k + 1], st);
        if (err == cudaSuccess) err = cudaStreamWaitEvent(hp.down, hp.ev[2 * k + 1], 0);
        if (err == cudaSuccess) err = cudaMemcpyAsync(y_host + off, y_dev + off, bytes, cudaMemcpyDeviceToHost, hp.down);
        if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host(D2H)");
    }
    err = cudaStreamSynchronize(hp.down);
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_host(sync)");
    return WPCD_OK;
}

wpcd_status wpcd_perm_apply_blocked_host(const wpcd_grid* g, const wpcd_channels* c, const int64_t* row_ptr_dev, const int32_t* geo_row_ptr_dev,
                                         const int32_t* col_idx_dev, const double* values_dev, const double* x_host, double* y_host,
                                         int n_vec, double* x_dev, double* y_dev, void* cuda_stream)
{
    if (!g || !c) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked_host: null handle");
    if (n_vec < 0) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked_host: negative size");
    const int64_t rows = wpcd_rows(g, c);
    if (rows == 0 || n_vec == 0) return WPCD_OK;
    if (!x_host || !y_host || !x_dev || !y_dev) return fail(WPCD_ERR_INVALID_ARG, "wpcd_perm_apply_blocked_host: null pointer");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t bytes = sizeof(double) * (size_t)rows * (size_t)n_vec;
    cudaError_t err = cudaMemcpyAsync(x_dev, x_host, bytes, cudaMemcpyHostToDevice, st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_blocked_host(H2D)");
    wpcd_status s = wpcd_perm_apply_blocked(g, c, row_ptr_dev, geo_row_ptr_dev, col_idx_dev, values_dev, x_dev, y_dev, n_vec, cuda_stream);
    if (s != WPCD_OK) return s;
    err = cudaMemcpyAsync(y_host, y_dev, bytes, cudaMemcpyDeviceToHost, st);
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_perm_apply_blocked_host(D2H)");
    return WPCD_OK;
}

wpcd_status wpcd_fp64_peak(void* cuda_stream, double* flops_out)
{
    if (!flops_out) return fail(WPCD_ERR_INVALID_ARG, "wpcd_fp64_peak: null pointer");
    cudaError_t err = run_fp64_peak(static_cast<cudaStream_t>(cuda_stream), flops_out);
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_fp64_peak");
    return WPCD_OK;
}

wpcd_status wpcd_trace_enable(int on)
{
    g_trace_on = on != 0;
    std::lock_guard<std::mutex> lock(g_trace_mutex);
    if (g_trace_on) {                       // have the timing events ready before the region that is timed
        while (g_trace_spare.size() < 2048) {
            cudaEvent_t e = nullptr;
            if (cudaEventCreate(&e) != cudaSuccess) break;
            g_trace_spare.push_back(e);
        }
    }
    return WPCD_OK;
}

wpcd_status wpcd_trace_read(double* ms_out, int64_t* launches_out)
{
    if (!ms_out) return fail(WPCD_ERR_INVALID_ARG, "wpcd_trace_read: null pointer");
    for (int i = 0; i < WPCD_TRACE_STAGES; ++i) { ms_out[i] = 0.0; if (launches_out) launches_out[i] = 0; }
    cudaError_t err = cudaSuccess;
    std::lock_guard<std::mutex> lock(g_trace_mutex);
    for (auto& r : g_trace) {
        float ms = 0.f;
        cudaError_t e = cudaEventSynchronize(r.e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.e0, r.e1);
        if (e != cudaSuccess) err = e;
        ms_out[r.stage] += ms;
        if (launches_out) launches_out[r.stage] += 1;
        if (g_trace_spare.size() < 4096) { g_trace_spare.push_back(r.e0); g_trace_spare.push_back(r.e1); }
        else { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    }
    g_trace.clear();
    if (err != cudaSuccess) return cuda_fail(err, "wpcd_trace_read");
    return WPCD_OK;
}

int64_t wpcd_launch_count(void) { return g_launches.load(); }

wpcd_status wpcd_debug_set(const char* key, int64_t value)
{
    if (!key) return fail(WPCD_ERR_INVALID_ARG, "wpcd_debug_set: null key");
    const std::string k(key);
    if (k == "spmv_lanes_per_row") g_debug.spmv_lanes_per_row = (int)value;
    else if (k == "spmv_no_pipeline") g_debug.spmv_no_pipeline = (int)value;
    else if (k == "no_pdl") g_debug.no_pdl = (int)value;
    else if (k == "chain_mode") g_debug.chain_mode = (int)value;
    else if (k == "blocked_tile_doubles") g_debug.blocked_tile_doubles = (int)value;
    else if (k == "blocked_no_mma") g_debug.blocked_no_mma = (int)value;
    else return fail(WPCD_ERR_INVALID_ARG, "wpcd_debug_set: unknown key " + k);
    return WPCD_OK;
}

}  // extern "C"
