"""The C-ABI library loads and exports every symbol include/pslmc.h declares; host logic; sharding."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1503_01725_b200 import build, binding
    build.build()
    return binding


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pslmc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b((?:psl|mc)_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(binding):
    names = declared_functions()
    assert set(names) == set(binding.EXPORTS), (names, binding.EXPORTS)
    L = binding.lib()
    for n in names:
        assert getattr(L, n) is not None
    syms = subprocess.check_output(["nm", "-D", "--defined-only", binding.LIB_PATH], text=True)
    for n in names:
        assert re.search(r"\bT %s\b" % n, syms), n


def test_struct_layouts_match_header(binding, tmp_path):
    """sizeof/offsetof from the real header (compiled with gcc) vs the ctypes mirror."""
    structs = {"psr_params_t": binding.psr_params_t, "jaws_t": binding.jaws_t, "phantom_t": binding.phantom_t,
               "beam_geom_t": binding.beam_geom_t, "mc_opts_t": binding.mc_opts_t, "mc_stats_t": binding.mc_stats_t}
    lines = []
    for name, st in structs.items():
        lines.append('printf("%s %%zu\\n", sizeof(%s));' % (name, name))
        for f, _ in st._fields_:
            lines.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (name, f, name, f))
    src = '#include <stdio.h>\n#include <stddef.h>\n#include "pslmc.h"\nint main(void){%s return 0;}' % "".join(lines)
    c = tmp_path / "layout.c"
    c.write_text(src)
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(c)])
    out = dict(l.split() for l in subprocess.check_output([str(exe)], text=True).splitlines())
    for name, st in structs.items():
        assert int(out[name]) == C.sizeof(st), name
        for f, _ in st._fields_:
            assert int(out["%s.%s" % (name, f)]) == getattr(st, f).offset, (name, f)


def test_no_cpu_fallback(binding, cfg):
    """Without a CUDA device the product path fails loudly (MC_E_CUDA) instead of computing on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    c = cfg("C0", False)
    with pytest.raises(binding.PslmcError) as e:
        binding.Psl(c["psr"], c["jaws"], c["n_sectors"])
    assert e.value.code == -4
    with pytest.raises(binding.PslmcError):
        binding.philox_debug(1, 2, 3, 4)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1503_01725_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "pslmc_oracle" not in txt, f
    assert "paper_1503_01725_b200" not in open(os.path.join(ROOT, "oracle", "pslmc_oracle.cpp")).read().replace(
        "paper_1503_01725_b200/csrc (the CUDA path)", "")
    assert not re.search(r"^\s*(import|from)\s+paper_1503_01725_b200", open(os.path.join(ROOT, "oracle", "__init__.py")).read(), flags=re.M)


def test_shard_range_partitions(binding):
    for N in (1, 7, 10_000_000):
        for world in (1, 2, 3, 8):
            r = [binding.shard_range(N, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == N
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1


WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r)
import numpy as np, torch, torch.distributed as dist
import oracle
from paper_1503_01725_b200 import binding, workloads
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%(port)d", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
c = workloads.make_config("C0")
psl = oracle.Psl(c["psr"], c["jaws"], c["n_sectors"]); ph = oracle.Phantom(c["phantom"])
N = 20000
a, b = binding.shard_range(N, rank, 2)
acc, res, _ = psl.dose(ph, c["beams"][0], N, 1, h_begin=a, h_end=b)
t = torch.from_numpy(acc)
dist.all_reduce(t, op=dist.ReduceOp.SUM)              # the one exchange of the multi-GPU path: int64 sum
led = torch.tensor([res["ledger"][k] for k in ("incident", "deposited", "escaped", "jaw")], dtype=torch.int64)
dist.all_reduce(led, op=dist.ReduceOp.SUM)
if rank == 0:
    full, fres, _ = psl.dose(ph, c["beams"][0], N, 1)
    assert np.array_equal(t.numpy(), full), "sharded sum differs"
    assert led.tolist() == [fres["ledger"][k] for k in ("incident", "deposited", "escaped", "jaw")]
    print("OK")
dist.destroy_process_group()
"""


def test_two_rank_sharding_is_bit_exact_gloo(tmp_path):
    """world_size-2 gloo run of the N>1 path's host logic: shard by history range, all-reduce the
    int64 tallies, compare bitwise with the unsharded run (the oracle stands in for the kernels)."""
    script = tmp_path / "worker.py"
    script.write_text(WORKER % dict(root=ROOT, port=29500 + os.getpid() % 2000))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert "OK" in outs[0][0]


def test_flag_and_error_constants_match_header(binding):
    """The binding's MC_FLAG_* / MC_ORDER_* values are the header's #defines (a mirror typed twice must not drift)."""
    import re
    text = open(os.path.join(ROOT, "include", "pslmc.h")).read()
    defs = {m.group(1): int(m.group(2)) for m in re.finditer(r"#define\s+(MC_[A-Z_0-9]+)\s+(-?\d+)", text)}
    flags = [k for k in defs if k.startswith("MC_FLAG_") or k.startswith("MC_ORDER_")]
    assert len(flags) >= 11
    for k in flags:
        assert getattr(binding, k) == defs[k], k
    assert defs["MC_E_WORKSPACE"] == -3 and defs["MC_E_OVERFLOW"] == -5 and defs["MC_OK"] == 0
    vals = [defs[k] for k in defs if k.startswith("MC_FLAG_")]
    assert len(set(vals)) == len(vals) and all(v & (v - 1) == 0 for v in vals)         # distinct single bits


def test_static_workspace_size_matches_header(binding):
    """mc_dose_static's scratch: the size the library reports is the header's MC_STATIC_WORKSPACE_BYTES (64 MiB), and the
    device image really holds an array of that size (a host-only query and an ELF look: no GPU needed)."""
    import re
    import subprocess
    text = open(os.path.join(ROOT, "include", "pslmc.h")).read()
    m = re.search(r"#define\s+MC_STATIC_WORKSPACE_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", text)
    assert m, "MC_STATIC_WORKSPACE_BYTES not found in pslmc.h"
    want = int(m.group(1)) << int(m.group(2))
    assert want == 64 << 20
    assert binding.lib().mc_static_workspace_bytes() == want
    elf = subprocess.run(["cuobjdump", "-elf", binding.LIB_PATH], capture_output=True, text=True)
    if elf.returncode == 0:                                   # (cuobjdump ships with the CUDA toolkit of this image)
        rows = [ln for ln in elf.stdout.splitlines() if "g_static_workspace" in ln and hex(want) in ln.lower()]
        assert rows, "no %d-byte g_static_workspace symbol in the device ELF" % want
