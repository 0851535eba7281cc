"""Host-side checks of the C ABI (no GPU needed): libmhd.so loads, exports every symbol include/*.h
declare, validates its arguments and fails loudly without a device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1810_12707_b200 import build, binding
    build.build()
    return binding.lib()


def declared_symbols():
    inc = os.path.join(ROOT, "include")
    text = "".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mhd_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    from paper_1810_12707_b200 import binding
    names = declared_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), "libmhd.so does not export %s" % n
    assert sorted(binding.SYMBOLS) == names


def test_init_argument_validation(lib):
    h = C.c_void_p()
    two_pi = 6.283185307179586
    assert lib.mhd_init(C.byref(h), 48, two_pi, 5 / 3, 0.0, 0.0, 1e-3) == -1      # not a power of two
    assert lib.mhd_init(C.byref(h), 8, two_pi, 5 / 3, 0.0, 0.0, 1e-3) == -1       # below the minimum
    assert lib.mhd_init(C.byref(h), 2048, two_pi, 5 / 3, 0.0, 0.0, 1e-3) == -1    # above the maximum
    assert lib.mhd_init(C.byref(h), 32, -1.0, 5 / 3, 0.0, 0.0, 1e-3) == -1
    assert lib.mhd_init(C.byref(h), 32, two_pi, 1.0, 0.0, 0.0, 1e-3) == -1        # gamma must exceed 1
    assert lib.mhd_init(C.byref(h), 32, two_pi, 5 / 3, -0.1, 0.0, 1e-3) == -1
    assert lib.mhd_init(C.byref(h), 32, two_pi, 5 / 3, 0.0, 0.0, 0.0) == -1
    assert lib.mhd_init(C.byref(h), 32, two_pi, 5 / 3, 0.01, 0.01, 1e-3) == 0 and h.value
    # unbound context: every compute call refuses
    assert lib.mhd_step(h, 1) == -2
    ptrs = (C.c_void_p * 8)()
    assert lib.mhd_rhs(h, 0, ptrs) == -2
    assert lib.mhd_set_fields(h, 1, 0, ptrs) == -2
    assert b"mhd_bind" in lib.mhd_last_error(h)
    assert lib.mhd_set_option(h, 99, 0) == -1
    # retired option ids keep their old meaning out of reach (include/mhd_bench.h); the one-launch S5 switch has a fresh id
    assert lib.mhd_set_option(h, 7, 8) == -1 and lib.mhd_set_option(h, 10, 1) == -1
    assert b"retired" in lib.mhd_last_error(h)
    assert lib.mhd_set_option(h, 14, 2) == 0 and lib.mhd_set_option(h, 14, 3) == -1
    assert lib.mhd_alt_launch_count(h, 13) == 0 and lib.mhd_alt_launch_count(h, 14) == 0 and lib.mhd_alt_launch_count(h, 1) == -1
    assert lib.mhd_destroy(h) == 0


def test_workspace_sizes(lib):
    assert lib.mhd_workspace_bytes(48, 0) == 0
    b32, b64 = lib.mhd_workspace_bytes(32, 0), lib.mhd_workspace_bytes(64, 0)
    assert b32 >= 48 * 32 ** 3 * 8 and b64 >= 48 * 64 ** 3 * 8 and b64 < 9 * b32
    # 512^3 must fit a B200's 180 GB with room to spare
    assert lib.mhd_workspace_bytes(512, 0) < 80e9
    assert lib.mhd_nspec(32) == 29 and lib.mhd_nspec(256) == 223


def test_chunked_pipeline_sizes(lib):
    """Placement arithmetic of the out-of-core path (config 6, 1024^3): compact storage fits one B200 entirely;
    with the state and the work fields in pinned host memory the device part is a few GB of staging."""
    OOC, STATE, WORK = 1, 2, 4
    kc = 1024 // 3
    compact = (2 * kc + 1) ** 2 * ((kc + 1 + 7) // 8 * 8) * 16
    zfull = 1024 * (2 * kc + 1) * ((kc + 1 + 7) // 8 * 8) * 16
    all_dev = lib.mhd_workspace_bytes(1024, OOC)
    assert 16 * compact + 16 * zfull < all_dev < 120e9 and lib.mhd_pinned_bytes(1024, OOC) == 0
    t1 = lib.mhd_workspace_bytes(1024, OOC | STATE)
    assert 16 * zfull < t1 < all_dev and 16 * compact <= lib.mhd_pinned_bytes(1024, OOC | STATE) < 16 * compact + 16 * 256
    t2 = lib.mhd_workspace_bytes(1024, OOC | STATE | WORK)
    assert 0 < t2 < 16e9
    assert lib.mhd_pinned_bytes(1024, OOC | STATE | WORK) >= 16 * (compact + zfull)
    # the paper's scenario (512^3 on a 16 GB P100): fits a 16 GiB budget with everything on the host
    assert 0 < lib.mhd_workspace_bytes(512, OOC | STATE | WORK | (16384 << 8)) <= 16384 << 20
    assert lib.mhd_workspace_bytes(512, OOC | 0x80) == 0      # unknown flag bit
    # per-rank storage of the slab decomposition (MHD_FLAG_RANKS(g) = (g - 1) << 4): 1/g of the state, 2/g of the work arrays
    r8 = lib.mhd_workspace_bytes(1024, OOC | (7 << 4))
    assert (16 * compact + 2 * 16 * zfull) / 8 < r8 < (16 * compact + 2 * 16 * zfull) / 8 * 1.1 + 12e9 and r8 < all_dev / 3
    assert lib.mhd_workspace_bytes(1024, OOC | STATE | (7 << 4)) == 0     # per-rank storage lives in HBM
    assert lib.mhd_workspace_bytes(1024, (7 << 4)) == 0                   # needs the chunked pipeline
    assert lib.mhd_workspace_bytes(512, STATE) == 0           # placement without the chunked pipeline


def test_variants_set_before_binding_are_refused_out_of_core(lib):
    """The ABI allows mhd_init -> mhd_set_param / mhd_set_option -> mhd_bind(MHD_FLAG_OUT_OF_CORE): forcing and the
    stress-tensor variant are in-core only and must be refused at bind time, not silently dropped."""
    two_pi = 6.283185307179586
    lib.mhd_set_param.argtypes = [C.c_void_p, C.c_int, C.c_double]
    for setup in ("force", "stress"):
        h = C.c_void_p()
        assert lib.mhd_init(C.byref(h), 32, two_pi, 5 / 3, 0.01, 0.01, 1e-3) == 0
        if setup == "force":
            assert lib.mhd_set_param(h, 2, 0.25) == 0            # MHD_PARAM_FORCE_AMP
        else:
            assert lib.mhd_set_option(h, 12, 1) == 0             # MHD_OPT_STRESS
        n = lib.mhd_workspace_bytes(32, 1)
        assert lib.mhd_bind(h, C.c_void_p(256), n, None, 1, None, 0) == -1
        assert b"in-core" in lib.mhd_last_error(h)
        lib.mhd_destroy(h)


def test_bind_without_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    assert lib.mhd_init(C.byref(h), 16, 6.283185307179586, 5 / 3, 0.0, 0.0, 1e-3) == 0
    n = lib.mhd_workspace_bytes(16, 0)
    rc = lib.mhd_bind(h, C.c_void_p(256), n, None, 0, None, 0)
    assert rc == -4 and b"no CUDA device" in lib.mhd_last_error(h)
    lib.mhd_destroy(h)
    from paper_1810_12707_b200 import MHD
    with pytest.raises(RuntimeError):
        MHD(16)
