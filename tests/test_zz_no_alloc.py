"""qhap_cut_eval_static: the cut evaluation with its scratch in a static device array (no workspace, no allocation).

Collected last on purpose (the run uses `pytest -x`).  Checks the new entry point against the existing
qhap_cut_eval (integer work: bit-exact, the bar every cut test uses) and against the oracle, on two calls in a row whose
sizes and contents differ (the array keeps the previous call's contents), and that oversized problems are rejected.
"""
import numpy as np
import pytest

from paper_2603_25762_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback)"
    from paper_2603_25762_b200 import binding
    return binding


def test_cut_eval_static_matches_workspace_path_twice_in_a_row(B, oracle):
    import torch
    fr, _ = synth.make_config(0)
    rg = oracle.read_graph(fr)
    sg = oracle.snp_graph(fr, 10, 0.1)
    # two calls in a row per graph / mode: many replicas first, then fewer (ragged word, stale bits behind it) -- and back
    for g, modes in ((rg, (0, 1)), (sg, (2,))):
        dg = B.upload_csr(g)
        for mode in modes:
            w = g["w_fx"] if mode == 2 else oracle.read_weights(g, mode)
            for call, R in enumerate((200, 37, 200)):
                s = synth.random_spins(100 * mode + call, g["n"], R)
                sd = torch.from_numpy(s).cuda()
                cut = torch.full((R,), -7, dtype=torch.int64, device="cuda")          # preallocated outputs: the call allocates nothing
                en = torch.full((R,), -7, dtype=torch.int64, device="cuda")
                rcut, ren = B.qhap_cut_eval(dg, mode, sd)                             # existing path (caller workspace); also
                torch.cuda.synchronize()                                              # loads the kernels both paths share
                free0 = torch.cuda.mem_get_info()[0]
                launches0 = B.qhap_launch_count()
                B.qhap_cut_eval_static(dg, mode, sd, cut=cut, energy=en)
                torch.cuda.synchronize()
                assert B.qhap_launch_count() > launches0                              # the library's own kernels ran
                assert torch.cuda.mem_get_info()[0] == free0                          # no device memory taken or returned
                assert torch.equal(cut, rcut) and torch.equal(en, ren), (mode, call, R)
                ecut, een = oracle.cut_eval(g["row_ptr"], g["col"], w, s)
                assert np.array_equal(cut.cpu().numpy(), ecut) and np.array_equal(en.cpu().numpy(), een), (mode, call, R)


def test_cut_eval_static_rejects_sizes_beyond_the_static_array(B, oracle):
    import torch
    # 512 + 4 n ceil(R / 32) bytes of scratch: just inside and just beyond QHAP_CUT_STATIC_BYTES, on an edgeless graph
    n = 4096
    words_max = (B.QHAP_CUT_STATIC_BYTES - 512) // 4 // n
    g = B.Csr(n, 0, torch.zeros(n + 1, dtype=torch.int32, device="cuda"), torch.zeros(1, dtype=torch.int32, device="cuda"),
              torch.zeros(1, dtype=torch.int32, device="cuda"), torch.zeros(1, dtype=torch.int32, device="cuda"))
    R_ok, R_big = 32 * words_max, 32 * words_max + 1
    cut, en = B.qhap_cut_eval_static(g, 0, torch.ones((n, R_ok), dtype=torch.int8, device="cuda"))
    assert int(cut.abs().max()) == 0 and int(en.abs().max()) == 0
    with pytest.raises(B.QhapError) as ei:
        B.qhap_cut_eval_static(g, 0, torch.ones((n, R_big), dtype=torch.int8, device="cuda"))
    assert ei.value.status == B.QHAP_ERR_WORKSPACE and "QHAP_CUT_STATIC_BYTES" in str(ei.value)
    # and the entry point still works afterwards
    cut, _ = B.qhap_cut_eval_static(g, 0, torch.ones((n, 8), dtype=torch.int8, device="cuda"))
    assert int(cut.abs().max()) == 0
