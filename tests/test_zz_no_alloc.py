"""mc_dose_static (include/pslmc.h): the entry point that allocates nothing - its scratch is a static __device__ array
inside libpslmc - against mc_dose with a caller workspace.  Integer tally, so the bar is the one every identity test
here uses: the int64 grid, the dose and the ledgers are bit-identical.  Collected last on purpose (file name): the
suite runs with pytest -x.  Self-contained: passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_1503_01725_b200 import binding
    binding.lib()
    return binding


def run(B, fn, dph, beam, N, seed, batch, **opt):
    import torch
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    dose = torch.empty(dph.nvox, dtype=torch.float64, device="cuda")
    fn(dph, beam, N, seed, batch=batch, dose_out=dose, dose_acc=acc, **opt)
    torch.cuda.synchronize()
    return acc.cpu().numpy(), dose.cpu().numpy(), B.stats()


def test_static_scratch_matches_caller_workspace_on_two_calls_in_a_row(B, cfg):
    import torch
    assert B.lib().mc_static_workspace_bytes() == 64 << 20
    calls = (("C0", 100_000, 7, 1 << 14, {}),                              # three pipelines, several batches per pipeline
             ("C1", 300_000, 8, 1 << 16, dict(pipelines=1)),               # another phantom and model: the array holds the first call's contents
             ("C0", 60_000, 9, 5_000, dict(pipelines=2, order=B.MC_ORDER_MIXED)))
    psl, dph = {}, {}
    for name in ("C0", "C1"):
        c = cfg(name)
        psl[name] = B.Psl(c["psr"], c["jaws"], c["n_sectors"]); dph[name] = B.DevicePhantom(c["phantom"])
    want = [run(B, psl[n].dose, dph[n], cfg(n)["beams"][0], N, seed, batch, **opt) for n, N, seed, batch, opt in calls]
    B.aux_streams(); torch.cuda.synchronize()
    got = []
    for n, N, seed, batch, opt in calls:                                   # back to back, nothing in between
        got.append(run(B, psl[n].dose_static, dph[n], cfg(n)["beams"][0], N, seed, batch, **opt))
    for (n, N, seed, batch, opt), (acc, dose, st), (acc0, dose0, st0) in zip(calls, got, want):
        assert acc0.sum() > 0
        assert np.array_equal(acc, acc0), (n, seed)
        assert np.array_equal(dose, dose0), (n, seed)
        assert st["ledger"] == st0["ledger"] and st["n_hist"] == st0["n_hist"] and sum(st["n_hist"]) == N
        assert st["n_jaw_rejected"] == st0["n_jaw_rejected"]


def test_static_scratch_allocates_nothing_and_rejects_what_does_not_fit(B, cfg):
    import torch
    c = cfg("C0")
    g, dph, beam = B.Psl(c["psr"], c["jaws"], c["n_sectors"]), B.DevicePhantom(c["phantom"]), c["beams"][0]
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    B.aux_streams()
    g.dose_static(dph, beam, 20_000, 3, batch=1 << 13, dose_acc=acc)       # first use: module load, symbol address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for seed in (4, 5):
        g.dose_static(dph, beam, 20_000, seed, batch=1 << 13, dose_acc=acc)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    # beyond the static array: MC_E_WORKSPACE with the sizes in the message, and nothing was scored
    before = acc.clone()
    assert g.workspace_bytes(dph, 1 << 20) > (64 << 20)
    with pytest.raises(B.PslmcError) as e:
        g.dose_static(dph, beam, 20_000, 6, batch=1 << 20, dose_acc=acc)
    assert e.value.code == -3 and "MC_STATIC_WORKSPACE_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert torch.equal(acc, before)
    # a caller workspace is refused rather than silently ignored
    ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    o = B._opts(workspace=ws, dose_acc=acc, pipelines=1)
    import ctypes as C
    rc = B.lib().mc_dose_static(g.h, C.byref(dph.c), C.byref(B._beam(beam)), 1000, 1, 1 << 10, None, C.byref(o))
    assert rc == -1
