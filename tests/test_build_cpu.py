"""-m "not gpu": what ptxas makes of the engine kernel (nvcc cross-compiles without a GPU).

The dispatcher warp keeps a whole PCIe poll (32 registers) in flight while it processes the previous
batch; one spilled register there makes ptxas store the poll to local memory right after issuing it,
which waits for the PCIe round trip and silently undoes the overlap (request rate 10 -> 7 M/s, measured).
So: no spills, 96 registers (18 warps per CTA: five warps on two of the four sub-partitions), and the
instructions the design rests on are in the SASS."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2607_02630_b200", "csrc")


def _nvcc():
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        pytest.skip("nvcc not available")
    return exe


@pytest.fixture(scope="module")
def cubin(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("cubin") / "aesoff_kernels.cubin")
    cmd = [_nvcc(), "-O3", "-std=c++17", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a", "-Xptxas", "-v",
           "-cubin", "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", out, os.path.join(CSRC, "aesoff_kernels.cu")]
    p = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert p.returncode == 0, p.stdout
    return out, p.stdout


def test_engine_kernel_registers_and_spills(cubin):
    """96 registers (18 warps per CTA: five warps on two of the four sub-partitions).  ptxas may park a few
    loop-invariant words of the worker loop (slot addresses) in local memory and reload them once per unit, but nothing
    may spill inside the cipher's round loops, and the dispatcher's polls no longer live in registers at all (they are
    cp.async copies into shared memory: a spilled poll register used to undo the overlap of poll and processing)."""
    path, log = cubin
    m = re.search(r"Compiling entry function '\S*aesoff_engine_kernel\S*' for 'sm_100a'.*?"
                  r"(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads.*?Used (\d+) registers",
                  log, re.S)
    assert m, log
    stack, st, ld, regs = map(int, m.groups())
    assert st <= 16 and ld <= 16, "the engine kernel spills %d B (stores) / %d B (loads)" % (st, ld)
    assert regs <= 96, regs
    assert stack <= 64, stack
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([exe, "-sass", path], stdout=subprocess.PIPE, text=True).stdout
    ins = [(int(a, 16), t) for a, t in re.findall(r"/\*([0-9a-f]{4,})\*/\s+(.*?);", sass)]
    index = {a: i for i, (a, _) in enumerate(ins)}
    round_loops = 0
    for i, (a, t) in enumerate(ins):
        mm = re.search(r"BRA.*?0x([0-9a-f]+)", t)
        if mm and int(mm.group(1), 16) < a and int(mm.group(1), 16) in index:
            body = [x for _, x in ins[index[int(mm.group(1), 16)]:i + 1]]
            if len(body) < 300 and sum("LDS" in x for x in body) >= 60:      # a main-round loop: 64 lookups per pass
                round_loops += 1
                assert not any(re.search(r"\b(LDL|STL)\b", x) for x in body), "local-memory traffic inside a round loop"
                assert "cp.async" not in "".join(body)
    assert round_loops >= 2
    assert "LDGSTS" in sass                                                     # the polls: cp.async into shared memory


def test_sass_has_the_instructions_the_design_rests_on(cubin):
    path, _ = cubin
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([exe, "-sass", path], stdout=subprocess.PIPE, text=True).stdout
    n_lds = len(re.findall(r"\bLDS R\d+, \[R\d+(\+0x[0-9a-f]+)?\]", sass))
    n_prmt = len(re.findall(r"\bPRMT\b", sass))
    assert n_lds >= 400 and n_prmt >= 400, (n_lds, n_prmt)       # one PRMT-built address per table lookup
    assert re.search(r"LDG\.E\.128\.STRONG\.GPU", sass) and re.search(r"STG\.E\.128\.STRONG\.GPU", sass)  # L2-only 128-bit payload
    assert "MEMBAR.SC.SYS" in sass or "MEMBAR.ALL.SYS" in sass or "ERRBAR" in sass  # system-scope fence before the mailbox
    assert re.search(r"BAR\.ARV|BAR\.SYNC", sass)                    # the named barriers of the start-up overlap


def test_bitslice_circuit_is_what_the_generator_derives():
    """aesoff_bitslice.cuh is generated: the committed file must be exactly what gen_bitslice_sbox.py prints (the
    generator checks its derivation against the S-box definition for all 256 inputs before it prints anything)."""
    import sys

    gen = os.path.join(CSRC, "gen_bitslice_sbox.py")
    p = subprocess.run([sys.executable, gen], stdout=subprocess.PIPE, text=True, check=True)
    assert p.stdout == open(os.path.join(CSRC, "aesoff_bitslice.cuh")).read()
