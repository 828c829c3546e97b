// gf8_stream_host.cuh -- host side of the streaming codec engine (gf8_stream.cuh): plans keyed by the LAYER list of a
// batched call (never by caller pointers), per-call pointer tables patched into the device-side description by a
// tiny kernel (tensormap.replace), and the launch.  Included by gf8_api.cu after gf8_fast.cuh.
#pragma once
#include "gf8_fast.cuh"
#include "gf8_stream.cuh"
#include <time.h>

struct SPlan {
    std::vector<uint64_t> key;
    int nT = 0, n_p1 = 0, n_upd = 0, n_maps = 0, n_shapes = 0, grid = 0, tap = 0;
    gf8::st::STensor* d_T = nullptr;
    gf8::st::P1Item* d_p1 = nullptr;
    gf8::st::TileEnt* d_tiles = nullptr;     // one entry per update tile, in global tile order (tile u -> CTA u mod grid)
    CUtensorMap *d_maps = nullptr, *d_tmpl = nullptr;
    int* d_shape_of = nullptr;
    const void** d_ptrs = nullptr;
    uint32_t* d_sync = nullptr;            // SY_WORDS words per problem, then the pass-1 item counter
    uint8_t* d_arena = nullptr;            // P', Q^T, Q'^T, (S E_A)^T of every problem
    size_t sync_bytes = 0;
    // per-call pointer staging: two pinned buffers used in turn, each guarded by an event
    const void** h_ptrs[2] = {nullptr, nullptr};
    cudaEvent_t h_ev[2] = {nullptr, nullptr};
    int h_next = 0;
    std::vector<const void*> last;         // pointer table of the previous call (unchanged -> nothing to patch)
    uint64_t basis_epoch = 0;
};

namespace {

constexpr size_t S_MAX_PLANS = 16;
constexpr int S_PASS_LAG = 450;                      // update-list entries between a tensor's last pass-A tile and its first pass-B tile
constexpr long long S_LEAD_BYTES = 96ll << 20;       // pass-1 may lead the update by this much gradient (L2 residency)

void splan_free(SPlan* p) {
    if (!p) return;
    cudaFree(p->d_T); cudaFree(p->d_p1); cudaFree(p->d_tiles); cudaFree(p->d_maps); cudaFree(p->d_tmpl); cudaFree(p->d_shape_of);
    cudaFree((void*)p->d_ptrs); cudaFree(p->d_sync); cudaFree(p->d_arena);
    for (int q = 0; q < 2; ++q) {
        if (p->h_ptrs[q]) cudaFreeHost((void*)p->h_ptrs[q]);
        if (p->h_ev[q]) cudaEventDestroy(p->h_ev[q]);
    }
    delete p;
}

// BF16 tensor map of rank 2 or 3 (dims / strides innermost first; strides[0] is implied), 128 B swizzle, zero OOB fill.
gf8_status make_map_nd(gf8_ctx* c, CUtensorMap* out, const void* ptr, int rank, const uint64_t* dims, const uint64_t* strides_bytes,
                       const uint32_t* box) {
    cuuint64_t gdim[3], gstr[2];
    cuuint32_t bx[3], es[3] = {1, 1, 1};
    for (int i = 0; i < rank; ++i) { gdim[i] = dims[i]; bx[i] = box[i]; }
    for (int i = 0; i + 1 < rank; ++i) gstr[i] = strides_bytes[i];
    const CUresult r = ((EncodeTiledFn)c->encode_tiled)(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(ptr), gdim, gstr,
                                                        bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(c, GF8_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d), rank %d", (int)r, rank);
    return GF8_OK;
}
// row-major [rows][cols] BF16 matrix, boxes of 64 columns x box_rows rows
gf8_status make_map_2d(gf8_ctx* c, CUtensorMap* out, const void* ptr, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    const uint64_t dims[2] = {cols, rows}, str[1] = {cols * 2};
    const uint32_t box[2] = {64, box_rows};
    return make_map_nd(c, out, ptr, 2, dims, str, box);
}
// the same matrix seen as [cols / 64][rows][64]: one box = `nblk` 64-column blocks of box_rows rows, stacked in shared memory
gf8_status make_map_3d(gf8_ctx* c, CUtensorMap* out, const void* ptr, uint64_t rows, uint64_t cols, uint32_t box_rows, uint32_t nblk) {
    const uint64_t dims[3] = {64, rows, cols / 64}, str[2] = {cols * 2, 128};
    const uint32_t box[3] = {64, box_rows, nblk};
    return make_map_nd(c, out, ptr, 3, dims, str, box);
}

inline bool stream_eligible(const gf8_ctx* c, const LayerState& L, gf8_dtype dt, bool tap) {
    if (!c->use_stream) return false;          // opt-in (GF8_STREAM=1, read once in gf8_create): see DESIGN.md 5 for where it stands
    if (!L.tc_ok || dt != GF8_DT_BF16 || c->precision != GF8_PREC_FAST) return false;
    if ((L.in.used && L.in.kp != 64) || (L.out.used && L.out.kp != 64)) return false;
    if (L.desc.d_in % 64) return false;
    (void)tap;
    return true;
}

gf8_status splan_build(gf8_ctx* c, SPlan* p, const std::vector<int>& lay, bool tap) {
    using namespace gf8::st;
    const int nT = (int)lay.size();
    p->nT = nT; p->tap = tap ? 1 : 0;
    std::vector<STensor> T(nT);
    std::vector<CUtensorMap> maps;
    std::map<std::pair<const void*, int>, int> map_idx;
    gf8_status s = GF8_OK;
    auto smap = [&](const void* buf, uint64_t rows, uint64_t cols, int box_rows) -> int {
        auto key = std::make_pair(buf, box_rows);
        auto f = map_idx.find(key);
        if (f != map_idx.end()) return f->second;
        CUtensorMap mp;
        if (s == GF8_OK) s = make_map_2d(c, &mp, buf, rows, cols, (uint32_t)box_rows);
        maps.push_back(mp);
        map_idx[key] = (int)maps.size() - 1;
        return (int)maps.size() - 1;
    };
    // arena layout
    size_t arena = 0;
    auto take = [&](size_t bytes) { const size_t o = arena; arena += (bytes + 1023) / 1024 * 1024; return o; };
    std::vector<size_t> oPp(nT), oQt(nT), oQpt(nT), oSEA(nT);
    for (int i = 0; i < nT; ++i) {
        const LayerState& L = c->layers[lay[i]];
        const size_t m = L.desc.d_out, n = L.desc.d_in;
        oPp[i] = take(m * 64 * 2); oQt[i] = take(((m + 255) / 256) * 16384); oQpt[i] = take(n * 64 * 2); oSEA[i] = take(64 * 64 * 2);
    }
    void* q = nullptr;
    if (cudaMalloc(&q, arena) != cudaSuccess) { cudaGetLastError(); return fail(c, GF8_ERR_NOMEM, "stream plan arena (%zu bytes)", arena); }
    p->d_arena = (uint8_t*)q;
    std::map<std::pair<int, int>, int> shape_idx;
    std::vector<CUtensorMap> tmpl;
    std::vector<int> shape_of(nT);
    std::vector<P1Item> p1;
    long long byte_pos = 0;
    int upd = 0, gate_next = 0;
    for (int i = 0; i < nT && s == GF8_OK; ++i) {
        LayerState& L = c->layers[lay[i]];
        STensor& t = T[i];
        memset(&t, 0, sizeof(t));
        t.m = L.desc.d_out; t.n = L.desc.d_in; t.useA = L.in.used ? 1 : 0; t.useG = L.out.used ? 1 : 0;
        t.fmt = L.desc.fmt; t.mode = tap ? M_TAP : (L.desc.scaling == GF8_SCALE_TENSOR ? M_AMAX : M_BLOCK);
        t.tiles_n = (t.n + 127) / 128; t.n_tiles = ((t.m + 127) / 128) * t.tiles_n;
        t.nP = t.useA ? (t.m + 255) / 256 : 0; t.nQ = t.useG ? (t.n + 255) / 256 : 0; t.nQP = (t.useA && t.useG) ? t.nQ : 0;
        t.dep_idx = SY_QP;               // the last pass-1 stage of a tensor counts on SY_QP (Q' items; P / Q panels if one-sided)
        t.dep_target = (t.useA && t.useG) ? t.nQP : (t.useA ? t.nP : t.nQ);
        t.upd_start = upd; upd += t.n_tiles;
        t.Pp = (bf16*)(p->d_arena + oPp[i]); t.Spart = (float*)(p->d_arena + oQt[i]); t.Qpt = (bf16*)(p->d_arena + oQpt[i]);
        t.SEA = (bf16*)(p->d_arena + oSEA[i]);
        t.eA = L.in.e; t.eG = L.out.e;
        t.byte_pos = byte_pos;
        if (t.useA) {
            t.map_UAt = smap(L.in.Ut16, 64, t.n, 64); t.map_UA128 = smap(L.in.U16, t.n, 64, 128); t.map_UA256 = smap(L.in.U16, t.n, 64, 256);
            t.map_Pp128 = smap(t.Pp, t.m, 64, 128); t.map_Pp64 = smap(t.Pp, t.m, 64, 64);
        }
        if (t.useG) {
            t.map_UGt = smap(L.out.Ut16, 64, t.m, 64); t.map_UG128 = smap(L.out.U16, t.m, 64, 128);
            t.map_Qpt128 = smap(t.Qpt, t.n, 64, 128);
        }
        if (t.useA && t.useG) t.map_SEA = smap(t.SEA, 64, 64, 64);
        auto sk = std::make_pair(t.m, t.n);
        auto f = shape_idx.find(sk);
        if (f == shape_idx.end()) {
            CUtensorMap mp[3];
            // (templates carry the arena's address; patch_kernel replaces it with the caller's gradient pointer)
            if (s == GF8_OK) s = make_map_2d(c, &mp[0], p->d_arena, t.m, t.n, 256);
            if (s == GF8_OK) s = make_map_3d(c, &mp[1], p->d_arena, t.m, t.n, 64, 4);
            if (s == GF8_OK) s = make_map_3d(c, &mp[2], p->d_arena, t.m, t.n, 128, 2);
            shape_idx[sk] = (int)shape_idx.size();
            f = shape_idx.find(sk);
            tmpl.insert(tmpl.end(), mp, mp + 3);
        }
        shape_of[i] = f->second;
        const long long bytes = (long long)t.m * t.n * 2;
        // lead control: the last tensor that lies wholly more than S_LEAD_BYTES of gradient behind this one must be complete
        while (gate_next < i && T[gate_next].byte_pos + (long long)T[gate_next].m * T[gate_next].n * 2 + S_LEAD_BYTES <= t.byte_pos) ++gate_next;
        const int gate = (tap || gate_next == 0) ? -1 : gate_next - 1, gate_total = gate >= 0 ? T[gate].n_tiles : 0;
        for (int i0 = 0; t.useA && i0 < t.m; i0 += 256) p1.push_back({K_PANEL_P, i, i0, std::min(256, t.m - i0), gate, gate_total, 0, 0});
        for (int j0 = 0; t.useG && j0 < t.n; j0 += 256) p1.push_back({K_PANEL_Q, i, j0, std::min(256, t.n - j0), gate, gate_total, 0, 0});
        byte_pos += bytes;
    }
    if (s != GF8_OK) return s;
    // dynamic maps follow the static ones
    const int n_static = (int)maps.size();
    for (int i = 0; i < nT; ++i) { T[i].map_src_p = n_static + 3 * i; T[i].map_src_q = n_static + 3 * i + 1; T[i].map_src_b = n_static + 3 * i + 2; }
    p->n_maps = n_static + 3 * nT; p->n_p1 = (int)p1.size(); p->n_upd = upd; p->n_shapes = (int)shape_idx.size();
    p->grid = std::max(1, std::min(c->num_sms, std::max(p->n_upd, p->n_p1)));
    // update list: pass-A tiles of a tensor, and its pass-B tiles S_PASS_LAG list entries later (by then the A tiles have run)
    std::vector<TileEnt> tiles;
    {
        std::vector<std::pair<int, size_t>> pendB;          // (tensor, list length when its A tiles were all listed)
        size_t headB = 0;
        auto emit = [&](int i, int pass) {
            for (int k = 0; k < T[i].n_tiles; ++k) tiles.push_back({i, (k / T[i].tiles_n) | ((k % T[i].tiles_n) << 16), pass, 0});
        };
        for (int i = 0; i < nT; ++i) {
            if (T[i].mode == M_AMAX) { emit(i, P_AMAX); pendB.push_back({i, tiles.size()}); }
            else emit(i, P_SINGLE);
            while (headB < pendB.size() && tiles.size() - pendB[headB].second >= (size_t)S_PASS_LAG) emit(pendB[headB++].first, P_CAST);
        }
        while (headB < pendB.size()) emit(pendB[headB++].first, P_CAST);
    }
    upd = (int)tiles.size();
    p->n_upd = upd;
    p->grid = std::max(1, std::min(c->num_sms, std::max(p->n_upd, p->n_p1)));
    p->sync_bytes = ((size_t)nT * SY_WORDS + 4) * sizeof(uint32_t);
    auto dm = [&](void** out, size_t bytes) -> bool { return cudaMalloc(out, std::max<size_t>(bytes, 16)) == cudaSuccess; };
    if (!dm((void**)&p->d_T, sizeof(STensor) * nT) || !dm((void**)&p->d_tiles, sizeof(TileEnt) * tiles.size()) || !dm((void**)&p->d_p1, sizeof(P1Item) * p1.size()) ||
        !dm((void**)&p->d_maps, sizeof(CUtensorMap) * p->n_maps) || !dm((void**)&p->d_tmpl, sizeof(CUtensorMap) * tmpl.size()) ||
        !dm((void**)&p->d_shape_of, sizeof(int) * nT) || !dm((void**)&p->d_ptrs, sizeof(void*) * 3 * nT) || !dm((void**)&p->d_sync, p->sync_bytes)) {
        cudaGetLastError();
        return fail(c, GF8_ERR_NOMEM, "stream plan tables");
    }
    for (int i = 0; i < nT; ++i) T[i].sync = p->d_sync + (size_t)i * SY_WORDS;
    CU_TRY(c, cudaMemcpy(p->d_T, T.data(), sizeof(STensor) * nT, cudaMemcpyHostToDevice));
    if (!tiles.empty()) CU_TRY(c, cudaMemcpy(p->d_tiles, tiles.data(), sizeof(TileEnt) * tiles.size(), cudaMemcpyHostToDevice));
    if (!p1.empty()) CU_TRY(c, cudaMemcpy(p->d_p1, p1.data(), sizeof(P1Item) * p1.size(), cudaMemcpyHostToDevice));
    if (n_static) CU_TRY(c, cudaMemcpy(p->d_maps, maps.data(), sizeof(CUtensorMap) * n_static, cudaMemcpyHostToDevice));
    CU_TRY(c, cudaMemcpy(p->d_tmpl, tmpl.data(), sizeof(CUtensorMap) * tmpl.size(), cudaMemcpyHostToDevice));
    CU_TRY(c, cudaMemcpy(p->d_shape_of, shape_of.data(), sizeof(int) * nT, cudaMemcpyHostToDevice));
    for (int b = 0; b < 2; ++b) {
        CU_TRY(c, cudaMallocHost((void**)&p->h_ptrs[b], sizeof(void*) * 3 * nT));
        CU_TRY(c, cudaEventCreateWithFlags(&p->h_ev[b], cudaEventDisableTiming));
    }
    return GF8_OK;
}

// Runs the eligible problems `idx` of a batched encode (or transform tap) through the streaming engine.
gf8_status stream_run(gf8_ctx* c, const std::vector<int>& idx, const int* layers, const void* const* grads, uint8_t* const* codes,
                      float* const* sinv, float* const* taps, cudaStream_t st) {
    using namespace gf8::st;
    const bool tap = taps != nullptr;
    std::vector<uint64_t> key;
    key.push_back(tap ? 2 : 1);
    for (int i : idx) key.push_back((uint64_t)layers[i]);
    SPlan* p = nullptr;
    for (SPlan* q : c->splans) if (q->key == key) { p = q; break; }
    if (!p) {
        GF_TRY(fast_init(c));
        if (!c->stream_attr_set) {
            CU_TRY(c, cudaFuncSetAttribute(stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, S_BYTES));
            c->stream_attr_set = true;
        }
        if (c->splans.size() >= S_MAX_PLANS) {            // evict the oldest plan (its work must have drained first)
            CU_TRY(c, cudaDeviceSynchronize());
            splan_free(c->splans.front());
            c->splans.erase(c->splans.begin());
        }
        p = new (std::nothrow) SPlan();
        if (!p) return fail(c, GF8_ERR_NOMEM, "host allocation failed");
        p->key = key;
        std::vector<int> lay;
        for (int i : idx) lay.push_back(layers[i]);
        const gf8_status s = splan_build(c, p, lay, tap);
        if (s != GF8_OK) { splan_free(p); return s; }
        c->splans.push_back(p);
    }
    // pointer table of this call; unchanged pointers (a training loop that reuses its buffers) need no patching
    std::vector<const void*> now(3 * (size_t)p->nT);
    for (int k = 0; k < p->nT; ++k) {
        const int i = idx[k];
        now[3 * k] = grads[i];
        now[3 * k + 1] = tap ? (const void*)taps[i] : (const void*)codes[i];
        now[3 * k + 2] = tap ? nullptr : (const void*)sinv[i];
    }
    if (now != p->last) {
        const int b = p->h_next;
        p->h_next ^= 1;
        CU_TRY(c, cudaEventSynchronize(p->h_ev[b]));      // (the copy that last used this staging buffer has run)
        memcpy((void*)p->h_ptrs[b], now.data(), sizeof(void*) * now.size());
        CU_TRY(c, cudaMemcpyAsync((void*)p->d_ptrs, (const void*)p->h_ptrs[b], sizeof(void*) * now.size(), cudaMemcpyHostToDevice, st));
        CU_TRY(c, cudaEventRecord(p->h_ev[b], st));
        patch_kernel<<<(p->nT + 127) / 128, 128, 0, st>>>(p->d_T, p->nT, p->d_ptrs, p->d_shape_of, p->d_tmpl, p->d_maps, p->tap);
        LAUNCH_CHECK(c);
        p->last.swap(now);
    }
    CU_TRY(c, cudaMemsetAsync(p->d_sync, 0, p->sync_bytes, st));
    int* ctr = reinterpret_cast<int*>(p->d_sync + (size_t)p->nT * SY_WORDS);
    stream_kernel<<<p->grid, S_THREADS, S_BYTES, st>>>(p->d_T, p->nT, p->d_p1, p->n_p1, p->n_upd, p->d_tiles, p->d_sync, p->d_maps, ctr, c->d_err, p->tap, c->d_prof);
    LAUNCH_CHECK(c);
#ifdef GF8_STREAM_PROF
    if (getenv("GF8_HEARTBEAT")) {   // debug builds only: where every warp is waiting 3 s after the launch (hang hunting)
        cudaStream_t s2; cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking);
        std::vector<long long> hb(32 * 160);
        struct timespec ts = {3, 0}; nanosleep(&ts, nullptr);
        cudaMemcpyAsync(hb.data(), c->d_prof + 16384, hb.size() * sizeof(long long), cudaMemcpyDeviceToHost, s2);
        cudaStreamSynchronize(s2);
        for (int b = 0; b < p->grid; ++b) {
            fprintf(stderr, "cta %3d:", b);
            for (int w = 0; w < 26; ++w) fprintf(stderr, " %lld", hb[(size_t)b * 32 + w]);
            fprintf(stderr, "\n");
        }
    }
    {   // debug builds only: average per-role wait profile of this launch (serialises the stream)
        std::vector<long long> h((size_t)p->grid * 64);
        cudaStreamSynchronize(st);
        cudaMemcpy(h.data(), c->d_prof, h.size() * sizeof(long long), cudaMemcpyDeviceToHost);
        if (getenv("GF8_TRACE")) {
            std::vector<long long> ev(4096);
            cudaMemcpy(ev.data(), c->d_prof + 20480, ev.size() * sizeof(long long), cudaMemcpyDeviceToHost);
            for (int cta = 0; cta < 2; ++cta) {
                const long long t0 = ev[cta * 2048 + 0];
                fprintf(stderr, "trace cta %d: tile | ready mma0 mma1 park0 park1 seen rel done cast0 cast1 (ns from first ready)\n", cta ? 77 : 0);
                for (int t = 0; t < 40; ++t) {
                    fprintf(stderr, "  %2d |", t);
                    for (int code : {0, 2, 3, 4, 5, 6, 7, 8, 9, 10}) fprintf(stderr, " %7lld", ev[cta * 2048 + code * 48 + t] - t0);
                    fprintf(stderr, "\n");
                }
            }
        }
        if (getenv("GF8_PERCTA")) {      // per-CTA: sready wait of the epilogue (role 3, slot 0) against pass-1 activity (role 4 total - waits; role 5 full wait)
            for (int b = 0; b < p->grid; ++b) {
                const long long* e = &h[((size_t)b * 8 + 3) * 8];
                const long long* pp = &h[((size_t)b * 8 + 4) * 8];
                const long long* pm = &h[((size_t)b * 8 + 5) * 8];
                const long long* um = &h[((size_t)b * 8 + 2) * 8];
                fprintf(stderr, "cta %3d: epi sready-wait %8lld ifull %8lld tfull %8lld | u-mma tempty %8lld full %8lld | p-prod gate %8lld dep %8lld pempty %8lld slack %8lld | p-mma idle %8lld\n", b, e[0], e[1], e[2],
                        um[1], um[3], pp[1], pp[2], pp[3], pp[5], pm[0]);
            }
        }
        const char* roles[7] = {"u-sched", "u-load", "u-mma", "u-epi0", "p-prod", "p-mma", "p-epi"};
        for (int r = 0; r < 7; ++r) {
            double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (int b = 0; b < p->grid; ++b) for (int q = 0; q < 8; ++q) a[q] += (double)h[((size_t)b * 8 + r) * 8 + q] / p->grid;
            fprintf(stderr, "stream prof %-7s %9.0f %9.0f %9.0f %9.0f %9.0f %9.0f %9.0f | total %9.0f cycles (avg / CTA)\n", roles[r], a[0], a[1], a[2], a[3],
                    a[4], a[5], a[6], a[7]);
        }
    }
#endif
    return GF8_OK;
}

}  // namespace
