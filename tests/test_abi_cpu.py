"""-m "not gpu": the C-ABI library builds, loads without a GPU, exports every function that
include/aesoff.h declares, and its host-side logic (key expansion = step a1, argument checks,
no-CPU-fallback behaviour) is right.  No compute call is made here.
"""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import oracle as o
from paper_2607_02630_b200 import build as aesoff_build
from paper_2607_02630_b200 import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    aesoff_build.build()
    import paper_2607_02630_b200.binding as B

    return B


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "aesoff.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"\b(aes_[a-z_0-9]+)\s*\(", text)
    return sorted(set(names))


def test_header_symbols_exported(P):
    names = _declared_functions()
    assert len(names) >= 15
    lib = ctypes.CDLL(P.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), "include/aesoff.h declares %s but libaesoff.so does not export it" % n
    assert set(names) == set(P.EXPORTS), "binding and header disagree: %s" % (set(names) ^ set(P.EXPORTS))


def test_no_torch_types_in_abi():
    text = open(os.path.join(ROOT, "include", "aesoff.h")).read()
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)  # declarations only, comments stripped
    assert "torch" not in code.lower() and "at::" not in code and "cudaStream_t" not in code
    assert set(re.findall(r"#include\s+<([^>]+)>", code)) == {"stddef.h", "stdint.h"}


def test_key_expansion_matches_oracle_and_fips_appendix_a(P, golden):
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 90]))
    keys = ([rng.bytes(16) for _ in range(50)] + [rng.bytes(24) for _ in range(50)] + [rng.bytes(32) for _ in range(50)]
            + [bytes(16), bytes(24), bytes(32), b"\xff" * 32])
    for key in keys:
        ctx = P.aes_ctx_create(key)
        rk, nr = P.aes_ctx_round_keys(ctx)
        P.aes_ctx_destroy(ctx)
        want, want_nr = o.key_expand(key)
        assert nr == want_nr and rk == want
    # the product's key schedule against the values PRINTED in FIPS-197 Appendix A.1 / A.3 directly
    g = golden("fips197_appendix_a.txt")
    ctx = P.aes_ctx_create(g["a1.key"])
    rk, nr = P.aes_ctx_round_keys(ctx)
    P.aes_ctx_destroy(ctx)
    assert nr == 10 and rk[16:32] == g["a1.w4_w7"] and rk[160:176] == g["a1.w40_w43"]
    ctx = P.aes_ctx_create(g["a2.key"])
    rk, nr = P.aes_ctx_round_keys(ctx)
    P.aes_ctx_destroy(ctx)
    assert nr == 12 and rk[24:28] == g["a2.w6"] and rk[192:208] == g["a2.w48_w51"]
    ctx = P.aes_ctx_create(g["a3.key"])
    rk, nr = P.aes_ctx_round_keys(ctx)
    P.aes_ctx_destroy(ctx)
    assert nr == 14 and rk[32:36] == g["a3.w8"] and rk[224:240] == g["a3.w56_w59"]


def test_ctx_errors(P):
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctx_create(bytes(20))
    assert e.value.code == P.AES_E_KEYBITS
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctx_create(bytes(16), keybits=100)
    assert e.value.code == P.AES_E_KEYBITS
    P.aes_ctx_destroy(0)  # NULL is a no-op


def test_fails_loudly_without_engine_or_gpu(P):
    """No CPU fallback: with no engine running a submit is AES_E_STOPPED; with no CUDA device the
    engine does not start."""
    try:
        import torch

        has_gpu = torch.cuda.is_available()
    except Exception:  # noqa: BLE001
        has_gpu = False
    ctx = P.aes_ctx_create(bytes(16))
    buf = (ctypes.c_uint8 * 64)()
    addr = (ctypes.addressof(buf) + 15) & ~15
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_submit(ctx, bytes(16), addr, addr, 16)
    assert e.value.code == P.AES_E_STOPPED
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_submit(ctx, bytes(16), addr + 1, addr + 1, 16)
    assert e.value.code == P.AES_E_ALIGN
    with pytest.raises(P.AesOffError) as e:
        P.aes_ctr_submit(ctx, bytes(16), addr, addr + 16, 32)
    assert e.value.code == P.AES_E_OVERLAP
    with pytest.raises(P.AesOffError) as e:
        P.aes_engine_stop()
    assert e.value.code == P.AES_E_STOPPED
    if not has_gpu:
        with pytest.raises(P.AesOffError) as e:
            P.aes_engine_start(0)
        assert e.value.code == P.AES_E_CUDA
        with pytest.raises(P.AesOffError) as e:
            P.aes_ctr_launch_batch([ctx], bytes(16), [addr], [addr], [16])
        assert e.value.code == P.AES_E_CUDA
    info = P.aes_engine_info()
    assert info["running"] == 0
    assert P.aes_strerror(P.AES_E_AGAIN) == "submission ring full"
    P.aes_ctx_destroy(ctx)


def test_engine_options_are_validated_before_any_cuda_call():
    """Bad option values are AES_E_INVAL whether or not there is a GPU: chunk_rows must be a power of two up to 64,
    at most 8 dispatcher warps, the ring a power of two in [64, 4096]."""
    import paper_2607_02630_b200.binding as P

    for kw in ({"chunk_rows": 3}, {"chunk_rows": 128}, {"n_dispatchers": 9}, {"ring_slots": 100}, {"ring_slots": 8192}):
        with pytest.raises(P.AesOffError) as e:
            P.aes_engine_start(0, **kw)
        assert e.value.code == P.AES_E_INVAL, kw


def test_product_does_not_touch_oracle():
    """The product path must not route through oracle/ (that would void parity)."""
    pkg = os.path.join(ROOT, "paper_2607_02630_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "aes_oracle" not in text, f
