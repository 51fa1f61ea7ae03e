// emulate.cpp — host emulation of the CUDA kernels (TEST INFRASTRUCTURE, CPU tests only).
//
// Compiles paper_2008_02478_b200/csrc/{kernels,apply_seq,khat_layout}.h with g++ and
// steps every kernel block by block, phase by phase, thread by thread — the same
// phase functions, launch sequence and kernel-spectrum layout the sm_100a build uses.
// It lets the index logic (digit-reversed orders, mirror rows, transposes, chunking)
// be checked against the oracle on a machine without a GPU.  libborisdemag.so does not
// contain or call any of this.
#include <cmath>
#include <cstring>
#include <limits>
#include <vector>

#include "../../paper_2008_02478_b200/csrc/apply_seq.h"

namespace {

// Thread order inside a phase: 0 ascending, 1 descending, 2 odd threads then even ones.  The threads of
// a phase must not depend on each other (only barriers order them), so every order has to give
// the same bits: a cheap stand-in for a race checker.
int g_thread_order = 0;

template <class K, int PH>
void run_phases(int bx, int by, const typename K::Args& a, float2* sm) {
    if (g_thread_order == 1) {
        for (int tid = K::NT - 1; tid >= 0; --tid) K::template phase<PH>(tid, bx, by, a, sm);
    } else if (g_thread_order == 2) {
        for (int tid = 1; tid < K::NT; tid += 2) K::template phase<PH>(tid, bx, by, a, sm);
        for (int tid = 0; tid < K::NT; tid += 2) K::template phase<PH>(tid, bx, by, a, sm);
    } else {
        for (int tid = 0; tid < K::NT; ++tid) K::template phase<PH>(tid, bx, by, a, sm);
    }
    if constexpr (PH + 1 < K::NPHASES) run_phases<K, PH + 1>(bx, by, a, sm);
}

struct HostLauncher {
    long launches = 0;
    template <class K>
    int run(bd::Grid g, const typename K::Args& a) {
        const long n = K::smem_elems(a);
        std::vector<float2> sm((size_t)n + 1);
        const float nan = std::numeric_limits<float>::quiet_NaN();
        for (unsigned by = 0; by < g.y; ++by)
            for (unsigned bx = 0; bx < g.x; ++bx) {
                for (auto& v : sm) { v.x = nan; v.y = nan; }     // shared memory starts undefined
                run_phases<K, 0>((int)bx, (int)by, a, sm.data());
            }
        ++launches;
        return 0;
    }
    // hooks of enqueue_apply: the emulation keeps everything in this one translation unit
    int tiled_2d(const bd::PlanView& p, const float* M, float* H) { return bd::dispatch_tiled_2d(*this, p, M, H); }
    int yfused3(const bd::PlanView& p) { return bd::enqueue_yfused3(*this, p); }
    int xz(const bd::PlanView& p, const float* M, float* H, bool fwd) { return bd::enqueue_xz<2, 256>(*this, p, M, H, fwd); }
    int plane_x(const bd::PlanView& p, const float* M, float* H, bool fwd) { return bd::enqueue_plane_x(*this, p, M, H, fwd); }
    int plane_yz(const bd::PlanView& p) { return bd::enqueue_plane_yz(*this, p); }
};

}  // namespace

namespace {
struct PlainPencil {           // one unpadded pencil in plain memory
    float2* p;
    static constexpr int off(int S, int r) { return r * S; }
    float2* ptr(int, int e) const { return p + e; }
    static float2 ld(const float2* q) { return *q; }
    void st(float2* q, float2 v) const { *q = v; }
    void pre(const float2*, int) const {}
    void stq(float2* q, float2 v, int) const { *q = v; }
};
template <int L, int P, bool INV>
void pk_pass_all(PlainPencil a, const float2* ptw) {
    constexpr int items = L / bd::dec_r(L, P);
    for (int it = 0; it < items; ++it) {
        if constexpr (!INV) bd::fwd_passM<L, P>(it, 0, 1, 1, a, a, ptw);
        else bd::inv_passM<L, P>(it, 0, 1, 1, a, a, ptw);
    }
}
}  // namespace


extern "C" {

// Kred: natural reduced spectrum [ncomp][nzr][nyr][nxr] in fp64 including the folded
// factor (as boris_demag_spectrum_host returns it).  M, H: fp32 [3][nz][ny][nx].
// cs_override > 0 forces the number of kx slots per chunk (to exercise chunking).
// nq_plane > 0: plane path with that many ky residues; 0: the plan's own choice; < 0: no plane path
int emu_apply_ex(int nx, int ny, int nz, const double* Kred, const float* M, float* H, int cs_override, int nq_plane);
// 1: the last kernel of the following emu_apply calls adds the field to H (BORIS_DEMAG_ACCUMULATE, fused)
static int g_emu_accumulate = 0;
void emu_set_accumulate(int on) { g_emu_accumulate = on; }
int emu_apply(int nx, int ny, int nz, const double* Kred, const float* M, float* H, int cs_override) {
    return emu_apply_ex(nx, ny, nz, Kred, M, H, cs_override, cs_override != 0 ? -1 : 0);
}
int emu_apply_ex(int nx, int ny, int nz, const double* Kred, const float* M, float* H, int cs_override, int nq_plane) {
    using namespace bd;
    LaunchCfg cfg = make_launch_cfg(nx, ny, nz);
    if (cs_override > 0) cfg.cs = cs_override;
    if (cs_override < 0) cfg.tiled = 0;          // force the untiled kernels
    if (nq_plane < 0) cfg.plane.on = 0;
    if (nq_plane > 0) cfg.plane = plane_geom(nx, ny, nz, nq_plane);
    if (nq_plane > 0 && !cfg.plane.on) return -1;
    const KLayout kl = cfg.tiled ? make_klayout_tiled(nx, ny, nz, cfg.cols) : make_klayout(nx, ny, nz, cfg.ty);
    const int Py = 2 * ny, Pz = nz > 1 ? 2 * nz : 1, NS = nx + 1;
    std::vector<float> Kst((size_t)kl.storage_elems());
    for (long i = 0; i < kl.storage_elems(); ++i) Kst[(size_t)i] = (float)storage_value(kl, i, Kred);
    std::vector<float2> twx((size_t)nx), twxp((size_t)nx / 2 + 1), twy((size_t)Py), twz((size_t)(Pz > 1 ? Pz : 1));
    fill_twiddles(twx.data(), nx, nx);
    fill_twiddles(twxp.data(), nx / 2 + 1, 2 * nx);
    fill_twiddles(twy.data(), Py, Py);
    if (nz > 1) fill_twiddles(twz.data(), Pz, Pz);
    const float nan = std::numeric_limits<float>::quiet_NaN();
    float2 poison; poison.x = nan; poison.y = nan;
    std::vector<float2> W((size_t)3 * NS * nz * ny, poison), T(nz > 1 ? (size_t)3 * cfg.cs * nz * Py : 1, poison);
    PlanView pv{nx, ny, nz, cfg, Kst.data(), twx.data(), twxp.data(), twy.data(), twz.data(), W.data(), T.data()};
    std::vector<float2> ptwx((size_t)ptw_total(nx)), ptwy((size_t)ptw_total(Py));
    fill_pass_twiddles(ptwx.data(), nx);
    fill_pass_twiddles(ptwy.data(), Py);
    std::vector<float2> V(cfg.tiled ? (size_t)3 * Pz * kl.ntl * ny * kl.cols : 1, bd_f2(0.f, 0.f));
    std::vector<float4> xpost((size_t)nx / 2 + 1);
    fill_xpost(xpost.data(), nx);
    pv.ptw_x = ptwx.data(); pv.ptw_y = ptwy.data(); pv.V = V.data(); pv.xpost = xpost.data();
    pv.en.accumulate = g_emu_accumulate;
    std::vector<float2> PX, PP, pltw, plzt;
    std::vector<float> KP;
    std::vector<int> kidx, slotky;
    if (cfg.plane.on) {
        const PlaneGeom& g = cfg.plane;
        const PlaneK pk = make_plane_k(nx, ny, nz, g);
        kidx.resize((size_t)g.nq * g.ls); slotky.resize((size_t)g.nq * g.nsl);
        plane_fill_tables(ny, g, kidx.data(), slotky.data());
        KP.resize((size_t)pk.storage_elems());
        for (long i = 0; i < pk.storage_elems(); ++i) KP[(size_t)i] = (float)plane_storage_value(pk, i, slotky.data(), Kred);
        // round trip of the layout: every natural entry is found where plane_storage_index_of says
        for (int c = 0; c < 6; ++c)
            for (int kz = 0; kz <= nz; ++kz)
                for (int ky = 0; ky <= ny; ++ky)
                    for (int kx = 0; kx <= nx; kx += (nx > 8 ? nx / 4 : 1)) {
                        const long si = plane_storage_index_of(pk, kidx.data(), c, kz, ky, kx);
                        const double ref = Kred[(((long)c * (nz + 1) + kz) * (ny + 1) + ky) * (nx + 1) + kx];
                        if (si < 0 || si >= pk.storage_elems() || KP[(size_t)si] != (float)ref) return -200;
                    }
        PX.assign((size_t)3 * nz * (nx + 1) * ny, poison);
        PP.assign((size_t)g.nq * 3 * nz * (nx + 1) * g.lsp, poison);
        pltw.resize((size_t)g.nq * (g.ls / 16) * 16); plzt.resize((size_t)g.zs * 16);
        plane_fill_tw(pltw.data(), ny, g);
        plane_fill_zt(plzt.data(), nz, g);
        pv.X = PX.data(); pv.P = PP.data(); pv.KP = KP.data(); pv.kidx = kidx.data();
        pv.pl_tw = pltw.data(); pv.pl_zt = plzt.data();
    }
    HostLauncher run;
    const int rc = enqueue_apply(run, pv, M, H);
    if (rc) return rc;
    return (int)run.launches == apply_launch_count(nx, nz, cfg) ? 0 : -100;
}

// gather the natural reduced spectrum back out of the storage layout (round trip check)
int emu_storage_roundtrip(int nx, int ny, int nz, const double* Kred, double* out) {
    using namespace bd;
    const LaunchCfg cfg = make_launch_cfg(nx, ny, nz);
    const KLayout kl = cfg.tiled ? make_klayout_tiled(nx, ny, nz, cfg.cols) : make_klayout(nx, ny, nz, cfg.ty);
    std::vector<double> Kst((size_t)kl.storage_elems());
    for (long i = 0; i < kl.storage_elems(); ++i) Kst[(size_t)i] = storage_value(kl, i, Kred);
    for (int c = 0; c < kl.ncomp; ++c)
        for (int kz = 0; kz < kl.nzr(); ++kz)
            for (int ky = 0; ky < kl.nyr(); ++ky)
                for (int kx = 0; kx < kl.nxr(); ++kx) {
                    float sign;
                    const long s = storage_index_of(kl, c, kz, ky, kx, sign);
                    if (s < 0 || s >= kl.storage_elems()) return -1;
                    out[kl.reduced_index(c, kz, ky, kx)] = sign * Kst[(size_t)s];
                }
    return 0;
}

void emu_set_thread_order(int order) { g_thread_order = order; }
int emu_pos_of_freq(int L, int k) { return bd::pos_of_freq(L, k); }
int emu_freq_of_pos(int L, int p) { return bd::freq_of_pos(L, p); }
int emu_khat_rows(int L) { return bd::khat_rows(L); }
int emu_khat_row_of_f(int L, int f) { return bd::khat_row_of_f(L, f); }
int emu_khat_f_of_row(int L, int r) { return bd::khat_f_of_row(L, r); }
int emu_slot_to_f(int L, int s) { return bd::slot_to_f(L, s); }
int emu_f_to_slot(int L, int f) { return bd::f_to_slot(L, f); }
int emu_dec(int L, int what) { return what < 0 ? bd::dec_np(L) : bd::dec_r(L, what); }

// One forward + inverse pass chain on a single pencil, no multiply: x[0..L/2) -> X (digit
// reversed, length L) -> back to x[0..L/2) scaled by L.  Used to test the butterflies alone.
int emu_fft_roundtrip(int L, const float* in_ri, float* spec_ri, float* out_ri) {
    using namespace bd;
    std::vector<float2> tw((size_t)L), a((size_t)L), b((size_t)L);
    fill_twiddles(tw.data(), L, L);
    for (int i = 0; i < L / 2; ++i) { a[i].x = in_ri[2 * i]; a[i].y = in_ri[2 * i + 1]; }
    YArgs f{a.data(), b.data(), L, L, 0, 0, 1, 1, tw.data()};
    YArgs g{b.data(), a.data(), L, L, 0, 0, 1, 1, tw.data()};
    HostLauncher run;
    int rc = dispatch_len(L, [&](auto ic) { return run.template run<YPass<decltype(ic)::value, false>>(Grid{1, 1}, f); });
    if (rc) return rc;
    for (int i = 0; i < L; ++i) { spec_ri[2 * i] = b[i].x; spec_ri[2 * i + 1] = b[i].y; }
    rc = dispatch_len(L, [&](auto ic) { return run.template run<YPass<decltype(ic)::value, true>>(Grid{1, 1}, g); });
    if (rc) return rc;
    for (int i = 0; i < L / 2; ++i) { out_ri[2 * i] = a[i].x; out_ri[2 * i + 1] = a[i].y; }
    return 0;
}

// The packed-arithmetic passes of the tiled path (pk.h, yfused.h) on one pencil: x[0..L/2) -> X (digit
// reversed, length L) -> back to x[0..L/2) scaled by L, with the per-pass twiddle tables of fill_pass_twiddles.
int emu_fft_roundtrip_pk(int L, const float* in_ri, float* spec_ri, float* out_ri) {
    using namespace bd;
    std::vector<float2> ptw((size_t)ptw_total(L)), a((size_t)L, bd_f2(0.f, 0.f));
    fill_pass_twiddles(ptw.data(), L);
    for (int i = 0; i < L / 2; ++i) { a[i].x = in_ri[2 * i]; a[i].y = in_ri[2 * i + 1]; }
    const int rc = dispatch_len(L, [&](auto ic) {
        constexpr int LL = decltype(ic)::value;
        constexpr int NP = dec_np(LL);
        PlainPencil pp{a.data()};
        pk_pass_all<LL, 0, false>(pp, ptw.data());
        if constexpr (NP >= 2) pk_pass_all<LL, 1, false>(pp, ptw.data());
        if constexpr (NP >= 3) pk_pass_all<LL, 2, false>(pp, ptw.data());
        for (int i = 0; i < LL; ++i) { spec_ri[2 * i] = a[i].x; spec_ri[2 * i + 1] = a[i].y; }
        if constexpr (NP >= 3) pk_pass_all<LL, 2, true>(pp, ptw.data());
        if constexpr (NP >= 2) pk_pass_all<LL, 1, true>(pp, ptw.data());
        pk_pass_all<LL, 0, true>(pp, ptw.data());
        return 0;
    });
    if (rc) return rc;
    for (int i = 0; i < L / 2; ++i) { out_ri[2 * i] = a[i].x; out_ri[2 * i + 1] = a[i].y; }
    return 0;
}

}  // extern "C"
