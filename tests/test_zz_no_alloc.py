"""fstat_eval_batch_noalloc (include/fstat.h): the evaluation of fstat_eval_batch with its workspace in the library's
static 32 MiB device array, for callers that cannot cudaMalloc inside the call.  Collected last on purpose."""
import numpy as np
import pytest

import synthetic as syn

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2407_10797_b200 as fs
    from paper_2407_10797_b200 import build
    build.build()
    fs.load_library()
    return fs


def _case(cfg, n_part, P):
    ds = syn.make_dataset(cfg, None)
    par = syn.draw_particles(cfg)[:P].copy()
    return ds, ds.edges(n_part), par


@pytest.mark.parametrize("which", ["tiny_direct_kernel", "slice_interpolating_kernel"])
def test_noalloc_call_equals_the_existing_path_twice_in_a_row(fs, which):
    """Same kernels, same launch order, another workspace: F and F_k equal fstat_eval_batch's bit for bit (the tests'
    tolerance against the oracle is 1e-5; the existing path is checked against the oracle in tests/test_gpu_parity.py),
    on two calls in a row -- the second one finds the first one's contents in the scratch array -- with a batch that is
    not a multiple of 128 and one invalid particle; then a different batch size in between, and the first one again."""
    import torch
    if which == "tiny_direct_kernel":
        ds, edges, par = _case(syn.CONFIGS[0], 4, 61)
    else:
        cfg = syn.Config(22, "noalloc_slice", 2.5 * syn.YEAR_S, 0.0200, 0.0203, (8,), (300,), 3.5 * syn.YEAR_S, "wide")
        ds, edges, par = _case(cfg, 8, 300)
    par[7, 2] = 0.3                                        # eta > 1/4: flies, F = -inf
    assert fs.fstat_noalloc_scratch_bytes() == 32 << 20
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges) as plan:
        p = torch.as_tensor(par, device="cuda")
        p_small = torch.as_tensor(np.ascontiguousarray(par[:40]), device="cuda")
        F_ref, Fk_ref = fs.fstat_eval_batch(plan, p)                       # plan set-up: builds the segment tables
        F_ref_s, Fk_ref_s = fs.fstat_eval_batch(plan, p_small)
        torch.cuda.synchronize()
        if which == "slice_interpolating_kernel":
            bins, _ = fs.fstat_plan_level_bins(plan)
            assert bins[1:].sum() > 0
        # the first call on a device resolves the array's address (cudaGetSymbolAddress); with lazy module loading that is
        # also when the driver places the 32 MiB array: do it before looking at the free memory
        fs.fstat_eval_batch_noalloc(plan, p_small, torch.empty(40, dtype=torch.float64, device="cuda"), None)
        torch.cuda.synchronize()
        outs = []
        for q, n in ((p, par.shape[0]), (p, par.shape[0]), (p_small, 40), (p, par.shape[0])):
            F = torch.full((n,), 7.0, dtype=torch.float64, device="cuda")
            Fk = torch.full((n, plan.n_part), 7.0, dtype=torch.float64, device="cuda")
            outs.append((F, Fk))
        free0 = torch.cuda.mem_get_info()[0]
        for (F, Fk), q in zip(outs, (p, p, p_small, p)):
            fs.fstat_eval_batch_noalloc(plan, q, F, Fk)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0       # the calls took no device memory
        for i, (F, Fk) in enumerate(outs):
            Fr, Fkr = (F_ref_s, Fk_ref_s) if i == 2 else (F_ref, Fk_ref)
            assert torch.equal(F, Fr), i
            assert torch.equal(Fk, Fkr), i
        assert torch.isneginf(outs[0][0][7])
        # F only
        F = torch.empty(par.shape[0], dtype=torch.float64, device="cuda")
        fs.fstat_eval_batch_noalloc(plan, p, F, None)
        torch.cuda.synchronize()
        assert torch.equal(F, F_ref)


def test_noalloc_call_rejects_what_does_not_fit_or_is_not_set_up(fs):
    import torch
    ds, edges, par = _case(syn.CONFIGS[0], 4, 64)
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges) as plan:
        p = torch.as_tensor(par, device="cuda")
        F = torch.empty(64, dtype=torch.float64, device="cuda")
        with pytest.raises(fs.FstatError) as ei:           # no segment tables for this batch size yet
            fs.fstat_eval_batch_noalloc(plan, p, F, None)
        assert ei.value.status == 4 and "segment tables" in str(ei.value)
        fs.fstat_eval_batch(plan, p)
        fs.fstat_eval_batch_noalloc(plan, p, F, None)      # now they exist
        # a batch whose workspace exceeds the array: 16 384 particles x 33 work segments x 80 B = 43 MB
        big = torch.as_tensor(np.ascontiguousarray(np.tile(par, (256, 1))), device="cuda")
        Fb = torch.empty(big.shape[0], dtype=torch.float64, device="cuda")
        fs.fstat_eval_batch(plan, big, Fb, None)
        with pytest.raises(fs.FstatError) as ei:
            fs.fstat_eval_batch_noalloc(plan, big, Fb, None)
        assert ei.value.status == 4 and "bytes of workspace" in str(ei.value)
        bigger = torch.as_tensor(np.ascontiguousarray(np.tile(par, (257, 1))), device="cuda")
        Fb2 = torch.empty(bigger.shape[0], dtype=torch.float64, device="cuda")
        with pytest.raises(fs.FstatError) as ei:           # P > 16384
            fs.fstat_eval_batch_noalloc(plan, bigger, Fb2, None)
        assert ei.value.status == 4
        torch.cuda.synchronize()


def test_noalloc_call_can_be_captured_in_a_cuda_graph_and_replayed(fs):
    """What the entry point is for: the whole evaluation (prologue, stride selection, main kernels, epilogue) captured once
    into a CUDA graph and replayed on new parameters written into the same input buffer -- no allocation, no host work per
    replay.  The replays equal fstat_eval_batch on the same parameters bit for bit."""
    import torch
    cfg = syn.Config(22, "noalloc_slice", 2.5 * syn.YEAR_S, 0.0200, 0.0203, (8,), (300,), 3.5 * syn.YEAR_S, "wide")
    ds, edges, par = _case(cfg, 8, 256)
    par2 = par[::-1].copy()
    with fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges) as plan:
        p = torch.as_tensor(par, device="cuda")
        F_ref, Fk_ref = fs.fstat_eval_batch(plan, p)                       # set-up: segment tables of this batch size
        F_ref2, Fk_ref2 = fs.fstat_eval_batch(plan, torch.as_tensor(par2, device="cuda"))
        F = torch.empty(256, dtype=torch.float64, device="cuda")
        Fk = torch.empty((256, plan.n_part), dtype=torch.float64, device="cuda")
        fs.fstat_eval_batch_noalloc(plan, p, F, Fk)                        # resolves the scratch address before the capture
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            fs.fstat_eval_batch_noalloc(plan, p, F, Fk)                    # on torch's current (capturing) stream
        F.zero_(); Fk.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(F, F_ref) and torch.equal(Fk, Fk_ref)
        p.copy_(torch.as_tensor(par2))                                     # new particles, same buffers
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(F, F_ref2) and torch.equal(Fk, Fk_ref2)
        del g
