// rx_emul.cu -- runs the phases of the "rx" kernel family (csrc/nl_rx_kernels.cuh) on the CPU, thread by
// thread, over bounds- and hazard-checked arrays.  TEST INFRASTRUCTURE (tests/test_host_emulation.py builds
// it with nvcc as a host program and compares its output with the fp64 oracle).
//
// The device kernels call exactly these phase functions with __syncthreads() between them; here a phase is a
// loop over the thread index and a barrier is the end of the loop.  Every shared-memory and workspace access
// goes through Checked<T>, which aborts on
//   - an index outside the array,
//   - a read of a word nobody has written (uninitialised shared memory),
//   - a word written by one thread and read or written by another thread within the same phase
//     (a race the barrier placement does not cover),
// i.e. the findings memcheck / racecheck report for block-synchronous code (profiles/r02_sanitizer.md).
//
// usage: rx_emul <NX> <in.bin> <out.bin>      (NY = 64; binary layout documented in test_host_emulation.py)
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "../../paper_2209_06731_b200/csrc/nl_rx_kernels.cuh"

namespace emu {

int g_phase = 0, g_tid = 0;
const char* g_phase_name = "";

struct Shadow {
    int wphase = -1, wtid = -1;      // last write
    int rphase = -1, rtid = -1;      // last read (rtid = -2: several threads)
    bool written = false;
};

[[noreturn]] void die(const char* what, const char* arr, long i) {
    std::fprintf(stderr, "rx_emul: %s: array %s index %ld, phase %d (%s), thread %d\n", what, arr, i, g_phase, g_phase_name, g_tid);
    std::exit(3);
}

template <class T> struct Checked {
    T* base;
    long n;
    Shadow* sh;                      // one per 4-byte word
    const char* name;
    static constexpr int W = sizeof(T) / 4;
    void check(long i) const { if (i < 0 || i >= n) die("index out of bounds", name, i); }
    T read(long i) const {
        check(i);
        for (int w = 0; w < W; ++w) {
            Shadow& s = sh[i * W + w];
            if (!s.written) die("read of unwritten word", name, i);
            if (s.wphase == g_phase && s.wtid != g_tid) die("read of a word another thread wrote in this phase", name, i);
            if (s.rphase == g_phase) { if (s.rtid != g_tid) s.rtid = -2; } else { s.rphase = g_phase; s.rtid = g_tid; }
        }
        return base[i];
    }
    void write(long i, const T& v) const {
        check(i);
        for (int w = 0; w < W; ++w) {
            Shadow& s = sh[i * W + w];
            if (s.wphase == g_phase && s.wtid != g_tid) die("two threads write one word in this phase", name, i);
            if (s.rphase == g_phase && s.rtid != g_tid) die("write of a word another thread read in this phase", name, i);
            s.wphase = g_phase; s.wtid = g_tid; s.written = true;
        }
        base[i] = v;
    }
    // view of the same storage with another element type (float2 <-> float4)
    template <class U> Checked<U> as() const { return Checked<U>{reinterpret_cast<U*>(base), n * (long)sizeof(T) / (long)sizeof(U), sh, name}; }
    Checked<T> offset(long elems) const { return Checked<T>{base + elems, n - elems, sh + elems * W, name}; }
};

}  // namespace emu

namespace emu {   // found by argument-dependent lookup from the phase templates in namespace gx
template <class T> T ld(Checked<T> p, int i) { return p.read(i); }
template <class T> void st(Checked<T> p, int i, const T& v) { p.write(i, v); }
template <class T> const void* addr_of(Checked<T> p, int i) { p.check(i); return p.base + i; }
}  // namespace emu

using emu::Checked;

template <class T> struct Arr {
    std::vector<T> data;
    std::vector<emu::Shadow> sh;
    const char* name;
    Arr(size_t n, const char* nm) : data(n), sh(n * sizeof(T) / 4), name(nm) {}
    Checked<T> view() { return Checked<T>{data.data(), (long)data.size(), sh.data(), name}; }
    void mark_written() { for (auto& s : sh) s.written = true; }
    void forget() { for (auto& s : sh) s = emu::Shadow(); }
};

#define PHASE(NAME, BODY)                                   \
    do {                                                    \
        ++emu::g_phase; emu::g_phase_name = NAME;           \
        for (int tid = 0; tid < C::NT; ++tid) { emu::g_tid = tid; BODY; } \
    } while (0)

struct Header { int Nx, Ny, Nz, Nl, Nm, Ns, J, pad; float dkx, dky; };

template <class C> int run(const Header& h, FILE* fi, const char* outpath) {
    const int NK = C::NK;
    const size_t nG = (size_t)h.Ns * h.Nm * h.Nl * h.Nz * NK, nPhi = (size_t)h.Nz * NK;
    const size_t szj = (size_t)h.Ns * h.Nz * h.J;
    std::vector<float2> G(nG), Phi(nPhi), tw(C::NX);
    std::vector<float> M(szj * NK), T((size_t)h.J * h.Nl), Tinv((size_t)h.Nl * h.J);
    auto rd = [&](void* p, size_t bytes) { if (std::fread(p, 1, bytes, fi) != bytes) { std::fprintf(stderr, "short input\n"); std::exit(2); } };
    rd(G.data(), nG * 8); rd(Phi.data(), nPhi * 8); rd(M.data(), M.size() * 4); rd(T.data(), T.size() * 4);
    rd(Tinv.data(), Tinv.size() * 4); rd(tw.data(), (size_t)C::NX * 8);

    Arr<float4> dchi(szj * C::H * C::NX, "dchi");
    Arr<float2> bhat(szj * h.Nm * NK, "bhat");
    Arr<float2> out(nG, "out");
    Arr<unsigned char> smem(C::SMEM_BYTES, "smem");   // words tracked through the float2/float4 views
    Arr<float2> twx(C::NX, "twx");
    std::vector<float> Ti(Tinv.size());
    for (size_t i = 0; i < Ti.size(); ++i) Ti[i] = -Tinv[i];
    const float scale = (float)(1.0 / ((double)C::NX * C::NY));

    auto S = [&]() { return Checked<float2>{reinterpret_cast<float2*>(smem.data.data()), C::S_ELEMS, smem.sh.data(), "smem.S"}; };
    auto stage4 = [&]() { return Checked<float4>{reinterpret_cast<float4*>(smem.data.data()), C::STAGE_BYTES / 16, smem.sh.data(), "smem.stage"}; };
    auto W4 = [&]() { return Checked<float4>{reinterpret_cast<float4*>(smem.data.data() + C::S_ELEMS * 8), C::W4_ELEMS, smem.sh.data() + C::S_ELEMS * 2, "smem.W4"}; };

    // ---- chi planes kernel
    for (size_t unit = 0; unit < szj; ++unit) {
        smem.forget(); twx.forget();
        const int z = (int)((unit / h.J) % h.Nz);
        PHASE("chi: twiddles + M.Phi", {
            for (int i = tid; i < C::NX; i += C::NT) st(twx.view(), i, tw[i]);
            for (int i = tid; i < NK; i += C::NT) {
                const float2 f = Phi[(size_t)z * NK + i];
                const float m = M[unit * NK + i];
                st(S(), i, make_float2(f.x * m, f.y * m));
            }
        });
        PHASE("chi: x inverse pass 1", gx::rx_x_inverse_pass1<C>(tid, S(), W4(), twx.view(), h.dkx, h.dky));
        PHASE("chi: x inverse pass 2", gx::rx_x_inverse_pass2<C>(tid, W4()));
        PHASE("chi: rows", gx::rx_row_chi<C>(tid, W4(), dchi.view().offset((long)unit * C::H * C::NX)));
    }
    // ---- bracket kernel, units in launch order; the last node of each (s,m,z) does the inverse Laguerre sum
    std::vector<unsigned> count((size_t)h.Ns * h.Nm * h.Nz, 0u);
    const size_t lstride = (size_t)h.Nz * NK;
    for (size_t unit = 0; unit < szj * h.Nm; ++unit) {
        smem.forget(); twx.forget();
        const int m = (int)(unit % h.Nm);
        const size_t sj = unit / h.Nm;
        const int j = (int)(sj % h.J), z = (int)((sj / h.J) % h.Nz), s = (int)(sj / ((size_t)h.J * h.Nz));
        const float2* g0 = G.data() + ((size_t)(s * h.Nm + m) * h.Nl * h.Nz + z) * NK;
        PHASE("twiddles", { for (int i = tid; i < C::NX; i += C::NT) st(twx.view(), i, tw[i]); });
        for (int l0 = 0; l0 < h.Nl;) {
            const bool first = l0 == 0;
            const int nl = std::min(first ? C::CAP : C::CAP - 1, h.Nl - l0);
            // TMA bulk copies: the async proxy writes whole planes (single writer, ordered by the mbarrier)
            ++emu::g_phase; emu::g_phase_name = "TMA landing"; emu::g_tid = -1;
            for (int l = 0; l < nl; ++l)
                for (int i = 0; i < NK; ++i)
                    st(Checked<float2>{reinterpret_cast<float2*>(smem.data.data()), C::STAGE_BYTES / 8, smem.sh.data(), "smem.stage2"},
                           (first ? l : l + 1) * NK + i, g0[(size_t)(l0 + l) * lstride + i]);
            PHASE("combine", gx::rx_combine<C>(tid, stage4(), T.data() + (size_t)j * h.Nl, l0, nl, first));
            l0 += nl;
        }
        PHASE("x inverse pass 1", gx::rx_x_inverse_pass1<C>(tid, S(), W4(), twx.view(), h.dkx, h.dky));
        PHASE("x inverse pass 2", gx::rx_x_inverse_pass2<C>(tid, W4()));
        PHASE("rows", gx::rx_row_bracket<C>(tid, W4(), dchi.view().offset((long)sj * C::H * C::NX)));
        PHASE("x forward pass 1", gx::rx_x_forward_pass1<C>(tid, W4(), twx.view()));
        PHASE("x forward pass 2", gx::rx_x_forward_pass2<C>(tid, W4(), bhat.view().offset((long)unit * NK).template as<float4>(), scale));
        unsigned& c = count[((size_t)s * h.Nm + m) * h.Nz + z];
        const unsigned old = c++;
        if ((old + 1u) % (unsigned)h.J == 0u) {
            auto bh4 = bhat.view().offset((long)(((size_t)(s * h.Nz + z) * h.J) * h.Nm + m) * NK).template as<float4>();
            auto out4 = out.view().offset((long)((((size_t)(s * h.Nm + m) * h.Nl) * h.Nz + z) * NK)).template as<float4>();
            PHASE("inverse Laguerre", gx::rx_laguerre_inverse<C>(tid, bh4, h.Nm * C::NK2, out4, (int)(lstride / 2), Ti.data(), h.Nl, h.J));
        }
    }
    for (size_t i = 0; i < out.sh.size(); ++i)
        if (!out.sh[i].written) { std::fprintf(stderr, "rx_emul: out word %zu never written\n", i); return 4; }
    FILE* fo = std::fopen(outpath, "wb");
    if (!fo) return 5;
    std::fwrite(out.data.data(), 8, nG, fo);
    std::fclose(fo);
    std::printf("rx_emul: ok, %d phases, NX=%d NY=%d\n", emu::g_phase, C::NX, C::NY);
    return 0;
}

int main(int argc, char** argv) {
    if (argc != 3) { std::fprintf(stderr, "usage: rx_emul in.bin out.bin\n"); return 1; }
    FILE* fi = std::fopen(argv[1], "rb");
    if (!fi) return 1;
    Header h;
    if (std::fread(&h, sizeof(h), 1, fi) != 1) return 2;
    if (h.Ny != 64) { std::fprintf(stderr, "NY must be 64\n"); return 1; }
    int rc = 1;
    if (h.Nx == 64) rc = run<gx::RxCfg<64, 64, 8, 8, 64, 6>>(h, fi, argv[2]);
    else if (h.Nx == 128) rc = run<gx::RxCfg<128, 64, 8, 16, 128, 3>>(h, fi, argv[2]);
    else if (h.Nx == 192) rc = run<gx::RxCfg<192, 64, 12, 16, 192, 2>>(h, fi, argv[2]);
    else if (h.Nx == 256) rc = run<gx::RxCfg<256, 64, 16, 16, 256, 1>>(h, fi, argv[2]);
    else std::fprintf(stderr, "no instantiation for NX=%d\n", h.Nx);
    std::fclose(fi);
    return rc;
}
