"""Host logic of the library against the oracle, on the CPU (no GPU needed).

* the library's own tensor (fp64 Newell near + triangular-Gauss quadrature far) vs the
  oracle's extended-precision Newell tensor (two different methods: DESIGN.md R3);
* the library's cosine/sine-transform kernel spectrum vs the oracle's rfftn of the padded tensor;
* the kernel-spectrum storage layout (round trip);
* the CUDA kernels' phase code, launch sequence and index maps, stepped thread by thread
  by the host emulation in tests/emu (test infrastructure), vs the oracle field.
"""
import ctypes
import os
import sys

import numpy as np
import pytest

from oracle import newell
from oracle.demag_fft import demag_fft, kernel_spectrum, padded_shape
from paper_2008_02478_b200 import binding, build, workloads as W

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "emu"))
import build_emu  # noqa: E402


@pytest.fixture(scope="session")
def emu():
    build.build()
    lib = ctypes.CDLL(build_emu.build())
    return lib


def vp(a):
    return ctypes.c_void_p(a.ctypes.data)


@pytest.mark.parametrize("dims,h", [((40, 30, 6), (5.0, 4.0, 3.0)), ((64, 8, 1), (2.0, 2.0, 1.0)),
                                    ((300, 2, 2), (2.0, 2.0, 1.0)), ((24, 24, 24), (2.0, 2.0, 2.0)),
                                    ((4, 4, 80), (5.0, 5.0, 0.5))])
def test_library_tensor_agrees_with_oracle_tensor(dims, h):
    build.build()
    nx, ny, nz = dims
    lib_T = binding.tensor_host(nx, ny, nz, *h)
    ora_T = newell.newell_tensor_octant(nx, ny, nz, *h)
    # a mismatch above ~1e-10 anywhere is a bug in one of the two;
    # across the near/far seam both are good to ~1e-12
    assert np.abs(lib_T - ora_T).max() < 2e-11   # 300 cells away the ORACLE (x87 extended) is the noisier side
    tr = lib_T[0] + lib_T[1] + lib_T[2]
    tr[0, 0, 0] -= 1
    assert np.abs(tr).max() < 2e-12            # pin P1 on the library's tensor


@pytest.mark.parametrize("shape,h,images", [((1, 6, 5), (4.0, 3.0, 2.0), (3, 2, 0)), ((3, 4, 5), (2.0, 3.0, 1.0), (2, 0, 1)),
                                            ((2, 12, 20), (2.0, 2.0, 1.0), (4, 0, 0)), ((1, 16, 16), (4.0, 4.0, 1.0), (12, 12, 0))])
def test_library_image_summed_tensor_agrees_with_oracle(shape, h, images):
    """Periodic boundary conditions: the library's sum over copies (plan_math.h, Gauss-quadrature far
    field) against the oracle's (oracle/demag_pbc.py, x87 Newell everywhere)."""
    from oracle.demag_pbc import image_tensor_table
    build.build()
    nz, ny, nx = shape
    lib_T = binding.tensor_host(nx, ny, nz, *h, images=images)
    ora_T = image_tensor_table(shape, h, images)
    # one copy: 2e-11 as above; every further copy adds its own far-field error (library quadrature <= 3e-13 beyond 10 cells)
    copies = (2 * images[0] + 1) * (2 * images[1] + 1) * (2 * images[2] + 1)
    assert np.abs(lib_T - ora_T).max() < 2e-11 + 3e-13 * copies
    tr = lib_T[0] + lib_T[1] + lib_T[2]
    tr[0, 0, 0] -= 1
    assert np.abs(tr).max() < 1e-11
    assert np.abs(lib_T - binding.tensor_host(nx, ny, nz, *h)).max() > 1e-5          # the copies do change it


@pytest.mark.parametrize("shape,h", [((1, 8, 16), (5.0, 5.0, 3.0)), ((4, 6, 8), (5.0, 4.0, 3.0)),
                                     ((1, 64, 32), (2.0, 2.0, 1.0)), ((8, 16, 16), (2.0, 2.0, 1.0))])
def test_library_spectrum_agrees_with_oracle_spectrum(shape, h):
    build.build()
    nz, ny, nx = shape
    if ny & (ny - 1):
        ny = 8
        shape = (nz, ny, nx)
    K = binding.spectrum_host(nx, ny, nz, *h)
    Ko = kernel_spectrum(shape, h)
    Pz, Py, Px = padded_shape(shape)
    scale = -1.0 / (2.0 * Px * Py * Pz)
    for c in range(K.shape[0]):
        ref = Ko[c][:K.shape[1], :ny + 1, :nx + 1].real
        assert np.abs(K[c] / scale - ref).max() < 1e-9
    # pin P11 on the library's spectrum: trace == 1 at every frequency (times the folded factor)
    assert np.abs((K[0] + K[1] + K[2]) / scale - 1).max() < 1e-10


@pytest.mark.parametrize("dims", [(8, 8, 1), (64, 128, 1), (16, 1024, 1), (8, 4, 2), (4, 16, 8), (4, 32, 64),
                                  (4, 512, 16), (4, 8, 128)])
def test_kernel_spectrum_storage_round_trip(emu, dims):
    nx, ny, nz = dims
    ncomp = 6 if nz > 1 else 4
    shape = (ncomp, nz + 1 if nz > 1 else 1, ny + 1, nx + 1)
    rng = np.random.default_rng(0)
    K = rng.standard_normal(shape)
    out = np.full(shape, np.nan)
    assert emu.emu_storage_roundtrip(nx, ny, nz, vp(K), vp(out)) == 0
    # entries that are their own mirror image must vanish for odd components; they do in
    # a real spectrum, so compare on a spectrum with that property
    assert np.array_equal(out, K)


def test_index_maps_are_bijections_and_rows_cover_the_half_spectrum(emu):
    for L in (4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048):
        pos = [emu.emu_pos_of_freq(L, k) for k in range(L)]
        assert sorted(pos) == list(range(L))
        assert all(emu.emu_freq_of_pos(L, p) == k for k, p in enumerate(pos))
        np_ = emu.emu_dec(L, -1)
        radices = [emu.emu_dec(L, p) for p in range(np_)]
        assert int(np.prod(radices)) == L
        RL, F = radices[-1], L // radices[-1]
        rows = emu.emu_khat_rows(L)
        assert rows == (F // 2 + 1 if F >= 2 else 1)
        fs = [emu.emu_khat_f_of_row(L, r) for r in range(rows)]
        assert sorted(fs) == list(range(rows))
        assert all(emu.emu_khat_row_of_f(L, f) == r for r, f in enumerate(fs))
        # every frequency 0..L/2 is stored in some (row, q), directly or through its mirror
        covered = set()
        for f in fs:
            for q in range(RL):
                k = f + F * q
                covered.add(min(k, L - k))
        assert covered == set(range(L // 2 + 1))


@pytest.mark.parametrize("core", ["emu_fft_roundtrip", "emu_fft_roundtrip_pk"])      # chunked kernels' core, packed core
@pytest.mark.parametrize("L", [4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048])
def test_pruned_forward_and_truncated_inverse_fft_against_numpy(emu, L, core):
    rng = np.random.default_rng(L)
    x = (rng.standard_normal(L // 2) + 1j * rng.standard_normal(L // 2)).astype(np.complex64)
    xin = np.ascontiguousarray(x.view(np.float32))
    spec = np.zeros(2 * L, np.float32)
    back = np.zeros(L, np.float32)
    assert getattr(emu, core)(L, vp(xin), vp(spec), vp(back)) == 0
    ref = np.fft.fft(np.concatenate([x.astype(np.complex128), np.zeros(L // 2)]))
    got = spec.view(np.complex64)
    pos = [emu.emu_pos_of_freq(L, k) for k in range(L)]
    assert np.abs(got[pos] - ref).max() < 3e-6 * np.abs(ref).max()
    assert np.abs(back.view(np.complex64) / L - x).max() < 3e-6


def test_kernel_tile_slots_are_a_bijection_onto_the_lower_half(emu):
    for L in (2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048):
        RL = emu.emu_dec(L, emu.emu_dec(L, -1) - 1)
        F = L // RL
        slots = [emu.emu_f_to_slot(L, f) for f in range(F // 2 + 1)]
        assert sorted(slots) == list(range(F // 2 + 1))
        assert all(emu.emu_slot_to_f(L, s) == f for f, s in enumerate(slots))


CASES = [
    # (nz, ny, nx), h, texture, cs_override
    ((1, 32, 32), (5.0, 5.0, 3.0), "random", 0),          # config C1 itself
    ((1, 4, 4), (5.0, 5.0, 3.0), "random", 0),
    ((1, 16, 64), (5.0, 4.0, 3.0), "vortex", 0),
    ((1, 1024, 4), (2.0, 2.0, 1.0), "random", 0),         # Py = 2048: three passes 16,16,8
    ((1, 512, 8), (2.0, 2.0, 1.0), "helix", 0),
    ((1, 128, 4), (2.0, 2.0, 1.0), "domains", 0),
    ((1, 4, 1024), (2.0, 2.0, 1.0), "random", 0),         # LX = 1024
    ((1, 8, 256), (4.0, 4.0, 4.0), "helix", 0),
    ((1, 16, 256), (3.0, 4.0, 2.0), "random", 0),         # 2-D mesh of 16 rows of 256: 8 rows per block
    ((16, 4, 256), (2.0, 3.0, 1.0), "random", 0),         # tiled 3-D, nz = 16 rows of 256: the same mapping with 512 threads
    ((2, 2, 4), (2.0, 2.0, 1.0), "random", 0),            # smallest 3-D mesh
    ((4, 8, 16), (5.0, 4.0, 3.0), "random", 0),
    ((8, 16, 8), (2.0, 2.0, 1.0), "random", 3),           # chunked kx slots with a ragged last chunk
    ((16, 32, 32), (2.0, 2.0, 1.0), "helix", 0),
    ((128, 4, 4), (2.0, 2.0, 2.0), "random", 0),          # Pz = 256 as in C4
    ((512, 2, 4), (2.0, 2.0, 2.0), "random", 0),          # Pz = 1024
    ((32, 512, 4), (2.0, 2.0, 1.0), "helix", 2),          # Py = 1024, Pz = 64 as in C5
    ((64, 4, 8), (2.0, 2.0, 1.0), "random", 0),           # z columns in 4 passes of 32 points
    ((256, 2, 4), (2.0, 2.0, 2.0), "random", 0),          # ... in 16 passes
    ((4, 8, 16), (5.0, 4.0, 3.0), "random", -1),          # chunked fallback kernels forced
    ((16, 32, 32), (2.0, 2.0, 1.0), "helix", -1),
]


@pytest.mark.parametrize("shape,h,texture,cs", CASES)
def test_emulated_kernels_match_the_oracle(emu, shape, h, texture, cs):
    nz, ny, nx = shape
    Ms = 8e5
    M = W.make_texture(texture, shape, Ms, seed=11)
    K = binding.spectrum_host(nx, ny, nz, *h)
    H = np.full(M.shape, np.nan, np.float32)
    assert emu.emu_apply(nx, ny, nz, vp(K), vp(M), vp(H), cs) == 0
    H_ref = demag_fft(M, h)
    err = np.abs(H - H_ref)
    assert err.max() <= 1e-5 * Ms                                   # north_star tolerance
    assert np.sqrt((err ** 2).sum() / (H_ref ** 2).sum()) <= 2e-6


@pytest.mark.parametrize("shape,cs", [((1, 16, 64), 0), ((1, 128, 8), 0), ((4, 8, 16), 0), ((32, 4, 32), 0),
                                      ((64, 4, 8), 0), ((8, 16, 8), -1)])
def test_phases_do_not_depend_on_the_order_of_their_threads(emu, shape, cs):
    """Threads of one phase may only meet at barriers: running them in another order must give the same bits."""
    nz, ny, nx = shape
    h = (2.0, 3.0, 1.0)
    M = W.make_texture("random", shape, 8e5, seed=17)
    K = binding.spectrum_host(nx, ny, nz, *h)
    out = []
    try:
        for order in (0, 1, 2):
            emu.emu_set_thread_order(order)
            H = np.full(M.shape, np.nan, np.float32)
            assert emu.emu_apply(nx, ny, nz, vp(K), vp(M), vp(H), cs) == 0
            out.append(H)
    finally:
        emu.emu_set_thread_order(0)
    assert np.isfinite(out[0]).all()
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])


# plane path (csrc/plane.h): nz = 32 slabs; nq = residues of ky (0: the plan's own choice)
PLANE_CASES = [
    ((32, 32, 4), (2.0, 2.0, 1.0), "random", 0),          # LS = 64, one residue (pruned first pass)
    ((32, 64, 8), (5.0, 4.0, 3.0), "random", 2),          # LS = 64, two residues
    ((32, 128, 4), (2.0, 2.0, 1.0), "helix", 4),          # LS = 64, four residues
    ((32, 128, 4), (2.0, 2.0, 1.0), "random", 2),         # LS = 128
    ((32, 128, 16), (2.0, 3.0, 1.0), "random", 0),        # LS = 256, one residue
    ((32, 256, 4), (2.0, 2.0, 1.0), "random", 0),         # LS = 256, two residues
    ((32, 512, 4), (2.0, 2.0, 1.0), "helix", 0),          # LS = 256, four residues: C5's y and z
    ((32, 256, 4), (2.0, 3.0, 1.0), "random", 8),         # LS = 64, eight residues
    ((32, 1024, 4), (2.0, 2.0, 1.0), "random", 0),        # LS = 256, eight residues (128th roots): ny = 1024
    ((16, 32, 8), (3.0, 2.0, 1.0), "random", 0),          # 16 cells: two lanes per column; LS = 64, one residue
    ((16, 128, 4), (2.0, 2.0, 1.0), "helix", 0),          # 16 cells, LS = 256
    ((16, 256, 4), (2.0, 2.0, 2.0), "random", 0),         # 16 cells, two residues
    ((8, 64, 8), (2.0, 3.0, 1.0), "random", 0),           # 8 cells: one lane, the transform itself pruned; LS = 128
    ((8, 512, 4), (2.0, 2.0, 1.0), "random", 0),          # 8 cells, four residues
    ((8, 128, 4), (4.0, 4.0, 1.0), "random", 4),          # 8 cells, LS = 64, four residues
    ((4, 64, 8), (2.0, 3.0, 1.0), "random", 0),           # 4 cells: one lane, 8 frequencies
    ((4, 512, 4), (2.0, 2.0, 1.0), "helix", 0),           # 4 cells, four residues
    ((2, 32, 16), (3.0, 2.0, 1.0), "random", 0),          # 2 cells: one lane, 4 frequencies
    ((2, 256, 4), (2.0, 2.0, 2.0), "random", 0),          # 2 cells, two residues
    ((4, 32, 256), (2.0, 2.0, 1.0), "random", 0),         # plane-path x kernels at LX = 256: 16-row blocks, three x passes
    ((64, 32, 4), (2.0, 2.0, 1.0), "random", 1),          # 64 cells: eight lanes per column; LS = 64
    ((64, 128, 4), (2.0, 3.0, 2.0), "helix", 2),          # 64 cells, LS = 128, two residues
]


@pytest.mark.parametrize("shape,h,texture,nq", PLANE_CASES)
def test_emulated_plane_path_matches_the_oracle(emu, shape, h, texture, nq):
    nz, ny, nx = shape
    Ms = 8e5
    M = W.make_texture(texture, shape, Ms, seed=13)
    K = binding.spectrum_host(nx, ny, nz, *h)
    H = np.full(M.shape, np.nan, np.float32)
    assert emu.emu_apply_ex(nx, ny, nz, vp(K), vp(M), vp(H), 0, nq) == 0
    H_ref = demag_fft(M, h)
    err = np.abs(H - H_ref)
    assert err.max() <= 1e-5 * Ms
    assert np.sqrt((err ** 2).sum() / (H_ref ** 2).sum()) <= 2e-6


def test_plane_path_phases_do_not_depend_on_thread_order(emu):
    shape, h = (32, 128, 4), (2.0, 3.0, 1.0)
    nz, ny, nx = shape
    M = W.make_texture("random", shape, 8e5, seed=19)
    K = binding.spectrum_host(nx, ny, nz, *h)
    out = []
    try:
        for order in (0, 1, 2):
            emu.emu_set_thread_order(order)
            H = np.full(M.shape, np.nan, np.float32)
            assert emu.emu_apply_ex(nx, ny, nz, vp(K), vp(M), vp(H), 0, 4) == 0
            out.append(H)
    finally:
        emu.emu_set_thread_order(0)
    assert np.isfinite(out[0]).all()
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])


@pytest.mark.parametrize("nx,ny,hx,hy,tk,ti,Z", [(24, 20, 5.0, 4.0, 4.9, 2.9, 4.5), (64, 8, 2.0, 2.0, 1.0, 1.0, 0.0),
                                                 (40, 40, 5.0, 5.0, 0.6, 4.9, -30.0), (16, 16, 3.0, 3.0, 2.0, 2.0, 2.0),
                                                 (200, 4, 2.0, 2.0, 1.0, 3.0, 2.5)])
def test_library_tensor_between_unequal_cuboids_agrees_with_oracle(nx, ny, hx, hy, tk, ti, Z):
    """Multi-layered convolution: csrc/ml_math.h (fp64 closed form near, Gauss quadrature of the dipole
    far) against oracle/multilayer.py (x87 closed form everywhere)."""
    from oracle.multilayer import pair_tensor_table
    build.build()
    lib_T = binding.ml_pair_tensor_host(nx, ny, hx, hy, tk, ti, Z)
    assert np.abs(lib_T - pair_tensor_table(nx, ny, hx, hy, tk, ti, Z)).max() < 2e-11


@pytest.mark.parametrize("shape,nq", [((1, 16, 64), 0), ((4, 8, 16), 0), ((32, 64, 8), 2)])       # XInvT, ZXInv, XInvP
def test_emulated_accumulate_adds_the_same_field_to_what_h_holds(emu, shape, nq):
    """BORIS_DEMAG_ACCUMULATE fused into the kernel that writes H (GRowsOutA / GRowsOutMapA): H0 + the plain result, bit for bit."""
    nz, ny, nx = shape
    h = (3.0, 2.0, 1.0)
    M = W.make_texture("random", shape, 8e5, seed=17)
    K = binding.spectrum_host(nx, ny, nz, *h)
    H = np.full(M.shape, np.nan, np.float32)
    assert emu.emu_apply_ex(nx, ny, nz, vp(K), vp(M), vp(H), 0, nq) == 0
    H0 = (np.random.default_rng(18).standard_normal(M.shape) * 1e4).astype(np.float32)
    Hacc = H0.copy()
    emu.emu_set_accumulate(1)
    try:
        assert emu.emu_apply_ex(nx, ny, nz, vp(K), vp(M), vp(Hacc), 0, nq) == 0
    finally:
        emu.emu_set_accumulate(0)
    assert np.array_equal(Hacc, H0 + H)


@pytest.fixture(scope="session")
def asan_emu():
    """tests/emu/asan_main.cpp: the emulation as an AddressSanitizer executable with exactly sized buffers."""
    import subprocess
    here = os.path.join(os.path.dirname(__file__), "emu")
    exe = os.path.join(here, "asan_emu")
    cuda_inc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "include")
    csrc = os.path.join(os.path.dirname(os.path.dirname(__file__)), "paper_2008_02478_b200", "csrc")
    deps = [os.path.join(here, f) for f in ("asan_main.cpp", "emulate.cpp")] + [os.path.join(csrc, f) for f in os.listdir(csrc) if f.endswith(".h")]
    if os.path.exists(exe) and all(os.path.getmtime(d) <= os.path.getmtime(exe) for d in deps):
        return exe
    # -O0: the instrumented template code compiles in half a minute (3.5 minutes at -O1) and still runs in seconds
    res = subprocess.run(["g++", "-std=c++17", "-O0", "-g", "-fsanitize=address", "-fno-omit-frame-pointer", "-I", cuda_inc,
                          "-I", here, "-o", exe, os.path.join(here, "asan_main.cpp")], capture_output=True, text=True)
    if res.returncode != 0:
        pytest.skip("no AddressSanitizer toolchain: " + res.stderr[-300:])
    return exe


# small-ny and small-nz shapes (more row groups than rows), every kernel path: tiled 2-D, tiled 3-D, plane (1, 2, 4, 8
# residues), chunked fallback
@pytest.mark.parametrize("args", [(8, 512, 4), (128, 256, 2), (64, 8, 1), (4, 2, 1), (16, 4, 8), (8, 4, 64), (4, 32, 32),
                                  (8, 64, 32, 0, 2), (4, 128, 32, 0, 4), (4, 256, 32, 0, 8), (8, 16, 8, -1), (16, 8, 4, 3),
                                  (8, 32, 16), (4, 64, 8), (8, 128, 16, 0, 2), (4, 32, 8, 0, -1), (4, 64, 64, 0, 1), (4, 128, 64, 0, 2), (8, 64, 4), (4, 32, 2), (8, 128, 2, 0, 2)])
def test_emulation_under_address_sanitizer(asan_emu, args):
    import subprocess
    res = subprocess.run([asan_emu] + [str(a) for a in args], capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, res.stdout[-500:] + res.stderr[-3000:]


@pytest.mark.parametrize("shape", [(16, 32, 32), (8, 32, 16), (32, 32, 8), (4, 32, 16), (2, 64, 8)])
def test_emulated_tiled_3d_kernels_on_slabs_the_plane_path_would_take(emu, shape):
    """XZFwd / YFused / ZXInv stay reachable (BORIS-internal choice: the plane path takes these slabs by default)."""
    nz, ny, nx = shape
    h, Ms = (2.0, 2.0, 1.0), 8e5
    M = W.make_texture("random", shape, Ms, seed=19)
    K = binding.spectrum_host(nx, ny, nz, *h)
    H = np.full(M.shape, np.nan, np.float32)
    assert emu.emu_apply_ex(nx, ny, nz, vp(K), vp(M), vp(H), 0, -1) == 0
    H_ref = demag_fft(M, h)
    err = np.abs(H - H_ref)
    assert err.max() <= 1e-5 * Ms and np.sqrt((err ** 2).sum() / (H_ref ** 2).sum()) <= 2e-6
