"""Host-side checks of the C-ABI library (no GPU needed): it builds, loads, exports every symbol that
include/acclb.h declares, sizes its workspace as DESIGN.md section 6 states, rejects bad arguments, and fails
loudly (never falls back) when there is no CUDA device."""
import ctypes as C
import re

import pytest

from paper_2505_01126_b200 import binding, build


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_symbols():
    text = binding.HEADER.read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(accLB_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert set(names) == set(binding.SYMBOLS), (names, binding.SYMBOLS)
    for name in names:
        assert hasattr(lib, name), f"libacclb.so does not export {name}"


def test_params_struct_matches_header():
    text = binding.HEADER.read_text()
    body = re.search(r"typedef struct \{(.*?)\} accLB_params;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"\b(?:double|int|void\*)\s+(\w+)(?:\[\d+\])?;", body)
    assert fields == [f[0] for f in binding.Params._fields_]


def test_workspace_bytes(lib):
    n = 32 ** 3
    a256 = lambda b: (b + 255) // 256 * 256
    small = a256(2 * 96 * 8) + a256(16 * 8)
    p = binding.make_params(tau=0.8)
    assert binding.workspace_bytes(32, 32, 32, p) == 2 * a256(27 * n * 8) + small
    p = binding.make_params(tau=0.8, store_fp32=1)
    assert binding.workspace_bytes(32, 32, 32, p) == 2 * a256(27 * n * 4) + small
    p = binding.make_params(tau=0.8, two_phase=1, mobility=0.05, sigma=0.01, host_staging=1)
    # seam strips of the 32 x 8 tile columns: u_x on 2 columns per tile column, u_y on 2 rows per tile row, u_z on 2
    # planes per z chunk (32^3: 1 tile column, 4 tile rows, chunks of 8 planes)
    seams = a256(32 * 32 * 2 * 1 * 8) + a256(32 * 2 * 4 * 32 * 8) + a256(2 * 4 * 32 * 32 * 8)
    # two population buffers, phi A / B, r, u (the unfused paths), seam strips, host staging
    assert binding.workspace_bytes(32, 32, 32, p) == (2 * a256(27 * n * 8) + 3 * a256(n * 8) + a256(3 * n * 8) + small
                                                      + seams + a256(5 * n * 8))
    p_rk = binding.make_params(tau=0.8, two_phase=1, mobility=0.05, sigma=0.01, host_staging=1, phi_rk3=1)
    assert binding.workspace_bytes(32, 32, 32, p_rk) == binding.workspace_bytes(32, 32, 32, p) + a256(n * 8)  # stage field
    # 512^3 two-phase fp64 fits one B200 (180 GB) with room to spare
    p = binding.make_params(tau=0.505, two_phase=1, mobility=0.05, sigma=0.02)
    assert 60e9 < binding.workspace_bytes(512, 512, 512, p) < 70e9


@pytest.mark.parametrize("shape,kw", [
    ((31, 32, 32), dict(tau=0.8)),            # nx odd
    ((2, 32, 32), dict(tau=0.8)),             # too thin
    ((32, 32, 32), dict(tau=0.5)),            # tau <= 1/2
    ((32, 32, 32), dict(tau=0.8, force_type=3)),
    ((32, 32, 32), dict(tau=0.8, two_phase=1, width=0.0)),
    ((32, 32, 32), dict(tau=0.8, two_phase=1, rho_g=0.0)),
    ((2048, 2048, 1024), dict(tau=0.8)),      # >= 2^31 nodes
    ((16384, 16384, 4), dict(tau=0.8)),       # 27 nx ny >= 2^32: in-slab offsets of the [z][i][y][x] layout are 32-bit
])
def test_invalid_arguments_give_zero_workspace(lib, shape, kw):
    assert binding.workspace_bytes(*shape, binding.make_params(**kw)) == 0


def test_create_rejects_bad_workspace_and_reports(lib):
    p = binding.make_params(tau=0.8)
    h = C.c_void_p()
    assert lib.accLB_create(C.byref(h), 32, 32, 32, C.byref(p), None, 0) == -2
    assert b"workspace" in lib.accLB_last_error()
    assert lib.accLB_create(C.byref(h), 31, 32, 32, C.byref(p), None, 0) == -1
    assert lib.accLB_create(C.byref(h), 32, 32, 32, C.byref(p), 0x1001, 1 << 40) == -2  # misaligned
    assert lib.accLB_step(None, 1) == -1 and lib.accLB_destroy(None) == -1


def test_no_cpu_fallback_without_gpu(lib):
    """On a box without a CUDA device create() must fail with ACCLB_ECUDA, not compute anything on the host."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present; covered by the gpu tests")
    p = binding.make_params(tau=0.8)
    h = C.c_void_p()
    # a fake, aligned, never-dereferenced address: create stops at cudaGetDeviceCount
    rc = lib.accLB_create(C.byref(h), 32, 32, 32, C.byref(p), 0x10000, 1 << 40)
    assert rc == -3 and not h.value
    with pytest.raises(Exception):
        binding.AccLB(32, 32, 32, tau=0.8)


def test_binding_and_product_do_not_touch_the_oracle():
    pkg = binding.HEADER.parent.parent / "paper_2505_01126_b200"
    for path in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")):
        text = path.read_text()
        assert "import oracle" not in text and "from oracle" not in text and "acclb_oracle" not in text, path
