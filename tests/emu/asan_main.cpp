// asan_main.cpp — the host emulation of the kernels (emulate.cpp) under AddressSanitizer with exactly sized M, H and
// kernel-spectrum buffers: an out-of-bounds access of any phase of any kernel path aborts the program.
// Test infrastructure (tests/test_host_logic.py builds and runs it); the values of the spectrum do not matter here.
//
//     asan_emu nx ny nz [cs_override nq_plane]
#include "emulate.cpp"

#include <cstdio>
#include <cstdlib>

int main(int argc, char** argv) {
    if (argc < 4) return 2;
    const int nx = atoi(argv[1]), ny = atoi(argv[2]), nz = atoi(argv[3]);
    const int cs = argc > 4 ? atoi(argv[4]) : 0, nq = argc > 5 ? atoi(argv[5]) : (cs != 0 ? -1 : 0);
    const size_t cells = (size_t)nx * ny * nz;
    const int nc = nz > 1 ? 6 : 4;
    const size_t nk = (size_t)nc * (nz > 1 ? nz + 1 : 1) * (ny + 1) * (nx + 1);
    std::vector<double> K(nk);
    for (size_t i = 0; i < nk; ++i) K[i] = 1e-9 * (double)((i * 2654435761u) % 1000);
    std::vector<float> M(3 * cells), H(3 * cells, 0.f);
    for (size_t i = 0; i < 3 * cells; ++i) M[i] = (float)((i * 40503u) % 2001) - 1000.f;
    const int rc = emu_apply_ex(nx, ny, nz, K.data(), M.data(), H.data(), cs, nq);
    double s = 0.0;
    for (float v : H) s += v;
    std::printf("rc %d checksum %.6e\n", rc, s);
    return rc == 0 && s == s ? 0 : 1;
}
