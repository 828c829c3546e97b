// gf8_stream_host.cuh -- host side of the streaming codec engine (gf8_stream.cuh): plans keyed by the LAYER list of a
// batched call (never by caller pointers), per-call pointer tables patched into the device-side description by a
// tiny kernel (tensormap.replace), and the launch.  Included by gf8_api.cu after gf8_fast.cuh.
#pragma once
#include "gf8_fast.cuh"
#include "gf8_stream.cuh"

struct SPlan {
    std::vector<uint64_t> key;
    int nT = 0, n_p1 = 0, n_upd = 0, n_maps = 0, n_shapes = 0, grid = 0, tap = 0;
    gf8::st::STensor* d_T = nullptr;
    gf8::st::P1Item* d_p1 = nullptr;
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
constexpr long long S_GROUP_BYTES = 24ll << 20;      // gradient bytes per pass-1 group
constexpr long long S_LEAD_BYTES = 72ll << 20;       // pass-1 may lead the update by this much gradient (L2 residency)

void splan_free(SPlan* p) {
    if (!p) return;
    cudaFree(p->d_T); cudaFree(p->d_p1); cudaFree(p->d_maps); cudaFree(p->d_tmpl); cudaFree(p->d_shape_of);
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
    if (!L.tc_ok || dt != GF8_DT_BF16 || c->precision != GF8_PREC_FAST) return false;
    if ((L.in.used && L.in.kp != 64) || (L.out.used && L.out.kp != 64)) return false;
    if (L.desc.d_in % 64) return false;
    const int64_t tiles = (int64_t)((L.desc.d_out + 127) / 128) * ((L.desc.d_in + 127) / 128);
    if (!tap && L.desc.scaling == GF8_SCALE_TENSOR && tiles > (int64_t)gf8::st::NPARK * c->num_sms) return false;
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
        oPp[i] = take(m * 64 * 2); oQt[i] = take(n * 64 * 4); oQpt[i] = take(n * 64 * 2); oSEA[i] = take(64 * 64 * 2);
    }
    void* q = nullptr;
    if (cudaMalloc(&q, arena) != cudaSuccess) { cudaGetLastError(); return fail(c, GF8_ERR_NOMEM, "stream plan arena (%zu bytes)", arena); }
    p->d_arena = (uint8_t*)q;
    std::map<std::pair<int, int>, int> shape_idx;
    std::vector<CUtensorMap> tmpl;
    std::vector<int> shape_of(nT);
    std::vector<P1Item> p1;
    std::vector<int> pend;                // tensors of the previous group: their S and Q' items follow this group's panels
    auto flush_pending = [&]() {
        for (int t : pend) if (T[t].useA && T[t].useG) p1.push_back({K_S, t, 0, 64});
        for (int t : pend) if (T[t].useA && T[t].useG)
            for (int j0 = 0; j0 < T[t].n; j0 += 256) p1.push_back({K_QP, t, j0, std::min(256, T[t].n - j0)});
        pend.clear();
    };
    long long byte_pos = 0, group_bytes = 0;
    int upd = 0;
    std::vector<int> cur;
    for (int i = 0; i < nT && s == GF8_OK; ++i) {
        LayerState& L = c->layers[lay[i]];
        STensor& t = T[i];
        memset(&t, 0, sizeof(t));
        t.m = L.desc.d_out; t.n = L.desc.d_in; t.useA = L.in.used ? 1 : 0; t.useG = L.out.used ? 1 : 0;
        t.fmt = L.desc.fmt; t.mode = tap ? M_TAP : (L.desc.scaling == GF8_SCALE_TENSOR ? M_PARK : M_BLOCK);
        t.tiles_n = (t.n + 127) / 128; t.n_tiles = ((t.m + 127) / 128) * t.tiles_n;
        t.nP = t.useA ? (t.m + 255) / 256 : 0; t.nQ = t.useG ? (t.n + 255) / 256 : 0; t.nQP = (t.useA && t.useG) ? t.nQ : 0;
        if (t.useA && t.useG) { t.dep_idx = SY_QP; t.dep_target = t.nQP; }
        else if (t.useA) { t.dep_idx = SY_P; t.dep_target = t.nP; }
        else { t.dep_idx = SY_Q; t.dep_target = t.nQ; }
        t.upd_start = upd; upd += t.n_tiles;
        t.Pp = (bf16*)(p->d_arena + oPp[i]); t.Qt = (float*)(p->d_arena + oQt[i]); t.Qpt = (bf16*)(p->d_arena + oQpt[i]);
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
        // pass-1 items of this tensor; a group is closed once it holds S_GROUP_BYTES of gradient
        const long long bytes = (long long)t.m * t.n * 2;
        if (group_bytes > 0 && group_bytes + bytes > S_GROUP_BYTES) {
            flush_pending();
            pend.swap(cur);
            group_bytes = 0;
        }
        for (int i0 = 0; t.useA && i0 < t.m; i0 += 256) p1.push_back({K_PANEL_P, i, i0, std::min(256, t.m - i0)});
        for (int j0 = 0; t.useG && j0 < t.n; j0 += 256) p1.push_back({K_PANEL_Q, i, j0, std::min(256, t.n - j0)});
        cur.push_back(i);
        group_bytes += bytes; byte_pos += bytes;
    }
    if (s != GF8_OK) return s;
    flush_pending();
    pend.swap(cur);
    flush_pending();
    // dynamic maps follow the static ones
    const int n_static = (int)maps.size();
    for (int i = 0; i < nT; ++i) { T[i].map_src_p = n_static + 3 * i; T[i].map_src_q = n_static + 3 * i + 1; T[i].map_src_b = n_static + 3 * i + 2; }
    p->n_maps = n_static + 3 * nT; p->n_p1 = (int)p1.size(); p->n_upd = upd; p->n_shapes = (int)shape_idx.size();
    p->grid = std::max(1, std::min(c->num_sms, std::max(p->n_upd, p->n_p1)));
    for (int i = 0; i < nT; ++i)
        if (T[i].mode == M_PARK && T[i].n_tiles > NPARK * p->grid) return fail(c, GF8_ERR_BAD_STATE, "stream plan: tensor too large to park");
    p->sync_bytes = ((size_t)nT * SY_WORDS + 4) * sizeof(uint32_t);
    auto dm = [&](void** out, size_t bytes) -> bool { return cudaMalloc(out, std::max<size_t>(bytes, 16)) == cudaSuccess; };
    if (!dm((void**)&p->d_T, sizeof(STensor) * nT) || !dm((void**)&p->d_p1, sizeof(P1Item) * p1.size()) ||
        !dm((void**)&p->d_maps, sizeof(CUtensorMap) * p->n_maps) || !dm((void**)&p->d_tmpl, sizeof(CUtensorMap) * tmpl.size()) ||
        !dm((void**)&p->d_shape_of, sizeof(int) * nT) || !dm((void**)&p->d_ptrs, sizeof(void*) * 3 * nT) || !dm((void**)&p->d_sync, p->sync_bytes)) {
        cudaGetLastError();
        return fail(c, GF8_ERR_NOMEM, "stream plan tables");
    }
    for (int i = 0; i < nT; ++i) T[i].sync = p->d_sync + (size_t)i * SY_WORDS;
    CU_TRY(c, cudaMemcpy(p->d_T, T.data(), sizeof(STensor) * nT, cudaMemcpyHostToDevice));
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
    stream_kernel<<<p->grid, S_THREADS, S_BYTES, st>>>(p->d_T, p->nT, p->d_p1, p->n_p1, p->n_upd, p->d_maps, ctr, c->d_err, S_LEAD_BYTES, p->tap);
    LAUNCH_CHECK(c);
    return GF8_OK;
}

}  // namespace
