"""CPU-only checks of the C-ABI boundary: libhypic.so builds, loads, exports every symbol include/hypic.h
declares, validates host-visible arguments before touching CUDA, and the binding has no CPU fallback."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hypic.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2607_01299_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hypic_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for required in ("hypic_segment_encode", "hypic_compose", "hypic_segment_encode_workspace",
                     "hypic_status_string", "hypic_version"):
        assert required in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2607_01299_b200 import binding
    names = declared_functions()
    assert names, "no functions parsed from the header"
    for name in names:
        assert hasattr(lib, name), f"libhypic.so does not export {name}"
    assert sorted(binding.EXPORTS) == names  # the binding mirrors the header, name for name


def test_version_and_status_strings(lib):
    from paper_2607_01299_b200 import binding
    assert binding.hypic_version() == 100
    seen = {binding.hypic_status_string(s) for s in range(5)}
    assert len(seen) == 5 and all(seen)
    assert binding.hypic_status_string(99) == "unknown status"


def test_argument_validation_needs_no_gpu(lib):
    """INVALID_ARG / UNSUPPORTED are decided from host-visible arguments before any CUDA call."""
    from paper_2607_01299_b200 import binding as b
    fake = ctypes.c_void_p(0x1000)  # never dereferenced: validation fails first
    enc = lib.hypic_segment_encode
    # null cu_seqlens
    assert enc(fake, fake, fake, fake, None, 1, 8, 1, 64, 64, 0, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    # negative sizes, bad enums
    assert enc(fake, fake, fake, fake, fake, -1, 8, 1, 64, 64, 0, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    assert enc(fake, fake, fake, fake, fake, 1, 8, 0, 64, 64, 0, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    assert enc(fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 7, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    assert enc(fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 5, fake, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    # null outputs / inputs
    assert enc(fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, None, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    assert enc(None, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    # misaligned pointer
    odd = ctypes.c_void_p(0x1004)
    assert enc(odd, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_INVALID_ARG
    # outside the built envelope
    assert enc(fake, fake, fake, fake, fake, 1, 8, 1, 96, 64, 0, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_UNSUPPORTED
    assert enc(fake, fake, fake, fake, fake, 1, 8, 1, 64, 4096, 0, 0, fake, fake, None, 0, None) == b.HYPIC_ERR_UNSUPPORTED

    comp = lib.hypic_compose
    assert comp(None, fake, fake, fake, None, 1, 4, 2, 1, 64, 64, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert comp(None, fake, fake, fake, fake, -1, 4, 2, 1, 64, 64, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert comp(None, None, fake, fake, fake, 1, 4, 2, 1, 64, 64, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert comp(None, fake, fake, fake, fake, 1, 4, 2, 1, 64, 64, None, None) == b.HYPIC_ERR_INVALID_ARG
    assert comp(None, fake, fake, fake, fake, 1, 4, 2, 1, 48, 64, fake, None) == b.HYPIC_ERR_UNSUPPORTED

    # the entry points added around the north-star pair validate the same way
    seam = lib.hypic_seam_window
    assert seam(fake, fake, fake, fake, fake, None, 1, 8, 1, 64, 64, 0, 0, None, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert seam(fake, fake, fake, fake, fake, fake, -1, 8, 1, 64, 64, 0, 0, None, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert seam(None, fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, None, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert seam(fake, fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, None, None, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert seam(fake, fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, odd, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert seam(fake, fake, fake, fake, fake, fake, 1, 8, 1, 80, 64, 0, 0, None, fake, fake, None) == b.HYPIC_ERR_UNSUPPORTED
    fwd = lib.hypic_forward_encode
    assert fwd(fake, fake, fake, fake, fake, None, 1, 8, 1, 64, 64, 0, 0, fake, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert fwd(fake, fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, None, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert fwd(fake, fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, fake, fake, None, None) == b.HYPIC_ERR_INVALID_ARG
    assert fwd(fake, fake, fake, fake, fake, fake, 1, 8, 1, 64, 64, 3, 0, fake, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    denc = lib.hypic_diag_encode
    assert denc(fake, fake, fake, None, 1, 8, 1, 64, 64, 0, 0, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert denc(fake, fake, fake, fake, 1, 8, 1, 64, 64, 0, 0, fake, None, None) == b.HYPIC_ERR_INVALID_ARG
    assert denc(fake, fake, None, fake, 1, 8, 1, 64, 64, 0, 0, fake, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert denc(fake, fake, fake, fake, 1, 8, 1, 96, 64, 0, 0, fake, fake, None) == b.HYPIC_ERR_UNSUPPORTED
    for dcomp in (lib.hypic_diag_compose, lib.hypic_diag_compose_f16):
        assert dcomp(None, fake, fake, fake, None, 1, 4, 2, 1, 64, 64, 0, fake, None) == b.HYPIC_ERR_INVALID_ARG
        assert dcomp(None, fake, None, fake, fake, 1, 4, 2, 1, 64, 64, 0, fake, None) == b.HYPIC_ERR_INVALID_ARG
        assert dcomp(None, fake, fake, fake, fake, 1, 4, 2, 1, 64, 64, 9, fake, None) == b.HYPIC_ERR_INVALID_ARG
        assert dcomp(None, fake, fake, fake, fake, 1, 4, 2, 1, 66, 64, 0, fake, None) == b.HYPIC_ERR_UNSUPPORTED
    assert lib.hypic_rope_compose_workspace(10, 128) == 10 * 128 * 4 and lib.hypic_rope_compose_workspace(0, 128) == 0
    for rc_ in (lib.hypic_rope_compose, lib.hypic_rope_compose_f16):
        big = 1 << 20
        assert rc_(None, fake, fake, fake, None, fake, fake, 1, 4, 2, 1, 64, 64, fake, fake, big, None) == b.HYPIC_ERR_INVALID_ARG
        assert rc_(None, fake, fake, fake, fake, None, fake, 1, 4, 2, 1, 64, 64, fake, fake, big, None) == b.HYPIC_ERR_INVALID_ARG
        assert rc_(None, fake, fake, fake, fake, fake, None, 1, 4, 2, 1, 64, 64, fake, fake, big, None) == b.HYPIC_ERR_INVALID_ARG
        assert rc_(None, fake, fake, fake, fake, fake, fake, 1, 4, 2, 1, 12, 64, fake, fake, big, None) == b.HYPIC_ERR_UNSUPPORTED
        assert rc_(None, fake, fake, fake, fake, fake, fake, 1, 4, 2, 1, 24, 64, fake, fake, big, None) == b.HYPIC_ERR_UNSUPPORTED
        assert rc_(None, fake, fake, fake, fake, fake, fake, 1, 4, 2, 1, 64, 64, fake, fake, 2 * 64 * 4 - 1, None) == b.HYPIC_ERR_WORKSPACE
        assert rc_(None, fake, fake, fake, fake, fake, fake, 1, 4, 2, 1, 64, 64, fake, None, 0, None) == b.HYPIC_ERR_WORKSPACE
    cf16 = lib.hypic_compose_f16
    assert cf16(None, fake, fake, fake, None, 1, 4, 2, 1, 128, 128, fake, None) == b.HYPIC_ERR_INVALID_ARG
    assert cf16(None, fake, fake, fake, fake, 1, 4, 2, 1, 64, 64, fake, None) == b.HYPIC_ERR_UNSUPPORTED
    assert lib.hypic_tuple_pack_f16(None, fake, 8, None) == b.HYPIC_ERR_INVALID_ARG
    assert lib.hypic_diag_encode_impl_for(1, 96, 64, 0, 0) == -b.HYPIC_ERR_UNSUPPORTED
    assert lib.hypic_diag_encode_impl_for(1, 128, 128, b.HYPIC_DT_BF16, 1) == b.HYPIC_IMPL_TENSOR
    assert lib.hypic_diag_encode_impl_for(1, 64, 64, b.HYPIC_DT_F32, 0) == b.HYPIC_IMPL_SIMT

    assert lib.hypic_set_impl(42) == b.HYPIC_ERR_INVALID_ARG
    assert lib.hypic_set_impl(b.HYPIC_IMPL_AUTO) == b.HYPIC_OK
    assert lib.hypic_segment_encode_workspace(-1, 0, 1, 64, 64, 0, 0) == 0


def test_binding_has_no_cpu_fallback(lib, monkeypatch):
    from paper_2607_01299_b200 import binding as b
    k = torch.zeros(4, 1, 64)
    cu = torch.tensor([0, 4], dtype=torch.int32)
    with pytest.raises(ValueError, match="CUDA tensor"):
        b.hypic_segment_encode(k, k.clone(), torch.zeros(4, 1), torch.zeros(4, 1), cu)
    E = torch.zeros(1, 1, 64, 64)
    with pytest.raises(ValueError, match="CUDA tensor"):
        b.hypic_compose(None, E, E.clone(), torch.zeros(1, dtype=torch.int32), torch.tensor([0, 1], dtype=torch.int32))
    # a missing library is a loud error, not a silent fallback
    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "LIB_PATH", os.path.join(ROOT, "no_such_dir", "libhypic.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        b.load_library()


def test_product_code_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_01299_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "hypic_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2607_01299_b200" not in text and "from paper_2607_01299_b200" not in text
