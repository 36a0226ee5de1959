// sanitize_main.cpp -- TEST INFRASTRUCTURE (tests/test_sanitizers.py): drives the host planner (csrc/planner.cpp) and the C
// oracle (oracle/mesh_attn_oracle.c) under AddressSanitizer + UndefinedBehaviorSanitizer (a host
// sanitizer build; compute-sanitizer is closed on the GPU pool).  The CUDA side of the library is not linked: the three
// symbols planner.cpp takes from capi.cu are stubbed here, so every plan is a host-only plan.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <string>
#include <vector>

#include "plan.hpp"

namespace mesh_attn {
static std::string g_err;
void set_error(const std::string& msg) { g_err = msg; }
int upload_plan(mesh_attn_plan*) { return MESH_ATTN_OK; }
void free_plan_device(mesh_attn_plan*) {}
}  // namespace mesh_attn

extern "C" {
int oracle_num_threads(void);
void oracle_attn_fwd_rows(const uint16_t*, const uint16_t*, const uint16_t*, int64_t, int, int, int, double, int, const int64_t*, const uint8_t*,
                          int64_t, const int64_t*, const int32_t*, double*, double*);
void oracle_attn_merge(int, int, const double*, const double*, double*, double*);
void oracle_attn_bwd_dq_rows(const uint16_t*, const uint16_t*, const uint16_t*, const uint16_t*, int64_t, int, int, int, double, int, const int64_t*,
                             int64_t, const int64_t*, const int32_t*, double*, double*, double*);
void oracle_attn_bwd_dkv_keys(const uint16_t*, const uint16_t*, const uint16_t*, const uint16_t*, int64_t, int, int, int, double, int, const int64_t*,
                              int64_t, const int64_t*, const double*, const double*, int64_t, const int64_t*, const int32_t*, double*, double*);
}

static int failures = 0;
#define CHECK(cond) do { if (!(cond)) { std::fprintf(stderr, "CHECK failed line %d: %s\n", __LINE__, #cond); ++failures; } } while (0)

static mesh_attn_plan_desc desc(int a, int b, int L, int hq, int hkv, int D, int causal, int kvr, int layout, int order, int kq, int kkv)
{
    mesh_attn_plan_desc d{};
    d.n = a * b; d.a = a; d.b = b; d.batch = 1; d.seq_total = a * b * L; d.heads_q = hq; d.heads_kv = hkv; d.head_dim = D;
    d.causal = causal; d.kvr = kvr; d.seq_layout = layout; d.order = order; d.k_q = kq; d.k_kv = kkv;
    return d;
}

static void exercise_plan(const mesh_attn_plan_desc& d)
{
    mesh_attn_plan* p = nullptr;
    CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_OK && p);
    if (!p) return;
    const int n = d.n;
    std::vector<int32_t> am((size_t)n * n);
    CHECK(mesh_attn_plan_am(p, am.data()) == MESH_ATTN_OK);
    std::vector<long> cells(n, 0);
    for (int32_t g : am) { CHECK(g >= 0 && g < n); if (g >= 0 && g < n) ++cells[g]; }
    for (int g = 0; g < n; ++g) CHECK(cells[g] == n);                       // every GPU owns exactly n cells
    std::vector<int32_t> iq(d.a), ikv(d.b);
    for (int g = 0; g < n; g += (n > 32 ? 7 : 1)) {
        CHECK(mesh_attn_plan_footprint(p, g, iq.data(), ikv.data()) == MESH_ATTN_OK);
        int32_t count = 0;
        CHECK(mesh_attn_plan_tiles(p, g, nullptr, 0, &count) == MESH_ATTN_EWORKSPACE);
        std::vector<int32_t> tiles((size_t)count * 4);
        CHECK(mesh_attn_plan_tiles(p, g, tiles.data(), count, &count) == MESH_ATTN_OK);
        for (int k = 0; k < count; ++k) CHECK(am[(size_t)tiles[4 * k] * n + tiles[4 * k + 1]] == g);
    }
    for (int pass = 0; pass < 2; ++pass) {
        int32_t count = 0;
        mesh_attn_plan_steps(p, pass, nullptr, 0, &count);
        std::vector<int32_t> steps((size_t)count * 4);
        CHECK(mesh_attn_plan_steps(p, pass, steps.data(), count, &count) == MESH_ATTN_OK);
        double mk, se, ex;
        CHECK(mesh_attn_plan_timeline(p, pass, &mk, &se, &ex) == MESH_ATTN_OK && mk <= se * (1 + 1e-9));
    }
    for (int what = 0; what <= 21; ++what) {
        int64_t v = -1;
        CHECK(mesh_attn_plan_query(p, what, &v) == MESH_ATTN_OK);
    }
    int64_t v = 0;
    CHECK(mesh_attn_plan_query(p, 99, &v) == MESH_ATTN_EINVAL);
    CHECK(mesh_attn_plan_query(p, MESH_ATTN_Q_HAS_DEVICE, &v) == MESH_ATTN_OK && v == 0);
    mesh_attn_plan_destroy(p);
}

static uint16_t bf16(double x)
{
    float f = (float)x;
    uint32_t u;
    std::memcpy(&u, &f, 4);
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

static void exercise_oracle(int causal, int striped)
{
    const int n = 3, L = 5, Hq = 4, Hkv = 2, D = 8;
    const int64_t N = n * L;
    std::vector<uint16_t> Q(N * Hq * D), K(N * Hkv * D), V(N * Hkv * D), dO(N * Hq * D);
    uint64_t s = 88172645463325252ull + causal * 7 + striped;
    auto rnd = [&]() { s ^= s << 13; s ^= s >> 7; s ^= s << 17; return (double)(s % 20001) / 10000.0 - 1.0; };
    for (auto& x : Q) x = bf16(rnd());
    for (auto& x : K) x = bf16(rnd());
    for (auto& x : V) x = bf16(rnd());
    for (auto& x : dO) x = bf16(rnd());
    std::vector<int64_t> pos(N);
    for (int p = 0; p < n; ++p) for (int r = 0; r < L; ++r) pos[p * L + r] = striped ? r * n + p : p * L + r;
    std::vector<int64_t> rows;
    std::vector<int32_t> heads;
    for (int64_t r = 0; r < N; ++r) for (int h = 0; h < Hq; ++h) { rows.push_back(r); heads.push_back(h); }
    const int64_t nq = (int64_t)rows.size();
    std::vector<double> O(nq * D), lse(nq), dQ(nq * D), lse2(nq), delta(nq);
    oracle_attn_fwd_rows(Q.data(), K.data(), V.data(), N, Hq, Hkv, D, 0.35, causal, pos.data(), nullptr, nq, rows.data(), heads.data(), O.data(), lse.data());
    // a key subset that leaves some rows without any visible key (reading R5)
    std::vector<uint8_t> sel(N, 0);
    for (int64_t t = N / 2; t < N; ++t) sel[t] = 1;
    std::vector<double> Op(nq * D), lsep(nq);
    oracle_attn_fwd_rows(Q.data(), K.data(), V.data(), N, Hq, Hkv, D, 0.35, causal, pos.data(), sel.data(), nq, rows.data(), heads.data(), Op.data(), lsep.data());
    for (auto& x : sel) x = !x;
    std::vector<double> Oq(nq * D), lseq(nq);
    oracle_attn_fwd_rows(Q.data(), K.data(), V.data(), N, Hq, Hkv, D, 0.35, causal, pos.data(), sel.data(), nq, rows.data(), heads.data(), Oq.data(), lseq.data());
    for (int64_t k = 0; k < nq; ++k) {                                         // merging the two halves gives the full row
        double parts[2 * D], lp[2] = {lsep[k], lseq[k]}, Om[D], lm;
        for (int d = 0; d < D; ++d) { parts[d] = Op[k * D + d]; parts[D + d] = Oq[k * D + d]; }
        oracle_attn_merge(2, D, parts, lp, Om, &lm);
        CHECK(std::fabs(lm - lse[k]) < 1e-12);
        for (int d = 0; d < D; ++d) CHECK(std::fabs(Om[d] - O[k * D + d]) < 1e-12);
    }
    oracle_attn_bwd_dq_rows(Q.data(), K.data(), V.data(), dO.data(), N, Hq, Hkv, D, 0.35, causal, pos.data(), nq, rows.data(), heads.data(), dQ.data(),
                            lse2.data(), delta.data());
    std::vector<double> lse_all((size_t)Hq * N), delta_all((size_t)Hq * N);
    for (int64_t k = 0; k < nq; ++k) { lse_all[heads[k] * N + rows[k]] = lse2[k]; delta_all[heads[k] * N + rows[k]] = delta[k]; CHECK(std::fabs(lse2[k] - lse[k]) < 1e-12); }
    std::vector<int64_t> qs(N), krows;
    std::vector<int32_t> kheads;
    for (int64_t r = 0; r < N; ++r) qs[r] = r;
    for (int64_t r = 0; r < N; ++r) for (int h = 0; h < Hkv; ++h) { krows.push_back(r); kheads.push_back(h); }
    std::vector<double> dK(krows.size() * D), dV(krows.size() * D);
    oracle_attn_bwd_dkv_keys(Q.data(), K.data(), V.data(), dO.data(), N, Hq, Hkv, D, 0.35, causal, pos.data(), N, qs.data(), lse_all.data(), delta_all.data(),
                             (int64_t)krows.size(), krows.data(), kheads.data(), dK.data(), dV.data());
    // sum_t dK[t] = 0 per KV head (rows of dS sum to zero)
    for (int h = 0; h < Hkv; ++h)
        for (int d = 0; d < D; ++d) {
            double acc = 0;
            for (size_t k = 0; k < krows.size(); ++k) if (kheads[k] == h) acc += dK[k * D + d];
            CHECK(std::fabs(acc) < 1e-10);
        }
    CHECK(oracle_num_threads() >= 1);
}

int main()
{
    // BASELINE.json configs[0..4] and structural variants
    exercise_plan(desc(2, 2, 256, 4, 4, 64, 0, 1, 0, 0, 1, 1));
    exercise_plan(desc(3, 3, 4096, 32, 32, 128, 0, 1, 0, 0, 1, 1));
    exercise_plan(desc(4, 4, 8192, 32, 32, 128, 1, 1, 1, 1, 2, 2));
    exercise_plan(desc(8, 8, 4096, 32, 8, 128, 1, 1, 1, 0, 1, 1));
    exercise_plan(desc(16, 16, 4096, 32, 32, 128, 1, 1, 1, 1, 2, 2));
    exercise_plan(desc(3, 5, 384, 4, 2, 128, 1, 0, 0, 1, 3, 1));
    exercise_plan(desc(5, 3, 128 * 16, 2, 1, 64, 1, 1, 1, 1, 1, 16));
    exercise_plan(desc(1, 4, 128 * 16, 2, 2, 64, 0, 0, 0, 1, 16, 1));
    {
        mesh_attn_plan_desc d = desc(2, 3, 256, 4, 2, 128, 1, 1, 1, 1, 2, 1);
        d.partial_mode = 1; d.batch = 3; d.precision = 1; d.tensor_layout = 1;
        exercise_plan(d);
        d = desc(2, 2, 256, 16, 8, 128, 0, 1, 0, 0, 1, 1);
        d.usp_lanes = 4; d.bwd_pairing = 2; d.bwd_piece_blocks = 2;
        exercise_plan(d);
        d.t_ag_kv = 1.f; d.t_ag_q = .5f; d.t_rs_q = .5f; d.t_c = .5f; d.gamma = 1.f; d.order = 1; d.k_q = d.k_kv = 1;
        exercise_plan(d);
    }
    // TAM example of the paper: 64 GPUs, a = b = 8, 8 per node: alpha 8 -> 112, alpha 4 -> 64
    {
        mesh_attn_plan_desc d = desc(8, 8, 128, 1, 1, 64, 0, 1, 0, 0, 1, 1);
        mesh_attn_plan* p = nullptr;
        CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_OK);
        int64_t q = 0, kv = 0;
        CHECK(mesh_attn_plan_tam_units(p, 8, 8, 0, &q, &kv) == MESH_ATTN_OK && q + kv == 112);
        CHECK(mesh_attn_plan_tam_units(p, 8, 4, 0, &q, &kv) == MESH_ATTN_OK && q + kv == 64);
        CHECK(mesh_attn_plan_tam_units(p, 8, 3, 0, &q, &kv) == MESH_ATTN_EINVAL);
        mesh_attn_plan_destroy(p);
    }
    // descriptors that must be refused, not crash
    {
        mesh_attn_plan* p = nullptr;
        mesh_attn_plan_desc d = desc(2, 2, 256, 4, 4, 64, 0, 1, 0, 0, 1, 1);
        d.n = 5; CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL && !p);
        d = desc(2, 2, 100, 4, 4, 64, 0, 1, 0, 0, 1, 1); CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL);
        d = desc(2, 2, 256, 4, 3, 64, 0, 1, 0, 0, 1, 1); CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL);
        d = desc(2, 2, 256, 4, 4, 96, 0, 1, 0, 0, 1, 1); CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EUNSUPPORTED);
        d = desc(2, 2, 256, 4, 4, 64, 0, 1, 0, 0, 5, 4); CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL);
        d = desc(2, 2, 256, 4, 4, 64, 0, 1, 0, 0, 1, 1); d.fwd_pairing = 2; CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL);
        d = desc(2, 2, 256, 4, 4, 64, 0, 1, 0, 0, 1, 1); d.out_dtype = 2; CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL);
        d = desc(2, 2, 256, 4, 4, 64, 0, 1, 0, 0, 1, 1); d.bwd_pairing = 7; CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL);
        d = desc(1, 4096, 2048, 1, 1, 64, 0, 1, 0, 0, 16, 1); d.partial_mode = 1; CHECK(mesh_attn_plan_create(&d, &p) == MESH_ATTN_EINVAL);
        CHECK(mesh_attn_plan_create(nullptr, &p) == MESH_ATTN_EINVAL);
        mesh_attn_plan_destroy(nullptr);
    }
    for (int causal = 0; causal < 2; ++causal)
        for (int striped = 0; striped < 2; ++striped) exercise_oracle(causal, striped);
    if (failures) { std::fprintf(stderr, "%d checks failed\n", failures); return 1; }
    std::puts("sanitize_main: ok");
    return 0;
}
