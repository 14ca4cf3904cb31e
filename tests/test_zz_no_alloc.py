"""lsp_periodogram_static: the entry point that allocates nothing (its workspace is a fixed 8 MiB `static __device__` array inside
the library; include/lsp.h).  Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.

Checked: its output against the existing path (lsp_periodogram, FP32-pipe form) and the fp64 oracle within the tolerance of
the other GPU tests, on calls in a row of DIFFERENT sizes (every call shares the one array, which keeps the previous call's
contents); at the maximum sizes, where the number of time splits is cut to what the array holds; that sizes beyond the limits are
refused with LSP_ELIMIT; that the device's free memory does not move across a call; and that a call can be captured into a CUDA
graph (a cudaMalloc under capture would fail it).  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-4          # north_star: max|P_gpu - P_ref| <= 1e-4 * max(P_ref)


def _existing(pkg, h, t, x, f_min, df, Nf):
    import torch
    h.set_param(pkg.PARAM_PIPE, pkg.PIPE_FP32)
    try:
        P, pi, pv = h.periodogram_batched(t.reshape(1, -1), x.reshape(1, -1), f_min, df, Nf)
        torch.cuda.synchronize()
    finally:
        h.set_param(pkg.PARAM_PIPE, 0)
    return P[0].cpu().numpy(), int(pi[0]), float(pv[0])


def _static(pkg, t, x, f_min, df, Nf):
    import torch
    P = torch.full((Nf,), -1.0, dtype=torch.float32, device="cuda")
    pi = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    pv = torch.full((1,), -7.0, dtype=torch.float32, device="cuda")
    pkg.periodogram_static(t, x, f_min, df, Nf, out=P, peak_idx=pi, peak_val=pv)
    torch.cuda.synchronize()
    return P.cpu().numpy(), int(pi[0]), float(pv[0])


def test_static_entry_point_matches_the_existing_path_on_calls_in_a_row(lsp):
    import torch
    pkg, h = lsp
    cases = [workloads.c2(), workloads.c1(), workloads.c2(), workloads.c1(Nt=777, Nf=4099, seed=31)]   # big, small, big, ragged
    free_after = []
    for n, w in enumerate(cases):
        t, x = torch.from_numpy(w.t).cuda(), torch.from_numpy(w.x).cuda()
        ref = oracle.periodogram(w.t, w.x, w.f_min, w.df, w.Nf)
        Pe, pie, pve = _existing(pkg, h, t, x, w.f_min, w.df, w.Nf)
        Ps, pis, pvs = _static(pkg, t, x, w.f_min, w.df, w.Nf)
        torch.cuda.synchronize()
        free_after.append(torch.cuda.mem_get_info()[0])
        top = float(ref.max())
        assert np.all(np.isfinite(Ps)) and Ps.shape == (w.Nf,)
        assert np.max(np.abs(Ps - Pe)) <= TOL * float(Pe.max()), "call %d against the existing path" % n
        assert np.max(np.abs(Ps - ref)) <= TOL * top, "call %d against the oracle" % n
        assert pis == int(np.argmax(Ps)) and pvs == float(Ps.max())
        assert pis == pie and ref[pis] >= (1.0 - 2 * TOL) * top     # the same peak as the existing path; the oracle's maximum to within the tolerance
        print("call %d (Nt=%d, Nf=%d): max |static - existing| = %.2e, |static - oracle| = %.2e of max P"
              % (n, w.Nt, w.Nf, np.max(np.abs(Ps - Pe)) / float(Pe.max()), np.max(np.abs(Ps - ref)) / top))
    # P only / peak only
    w = cases[1]
    t, x = torch.from_numpy(w.t).cuda(), torch.from_numpy(w.x).cuda()
    P_only = pkg.periodogram_static(t, x, w.f_min, w.df, w.Nf)
    torch.cuda.synchronize()
    assert np.array_equal(P_only.cpu().numpy(), _static(pkg, t, x, w.f_min, w.df, w.Nf)[0])      # (and run to run bit-identical)
    pi = torch.zeros(1, dtype=torch.int32, device="cuda"); pv = torch.zeros(1, dtype=torch.float32, device="cuda")
    lib = pkg.load()
    assert lib.lsp_periodogram_static(t.data_ptr(), x.data_ptr(), w.Nt, w.f_min, w.df, w.Nf, None, pi.data_ptr(), pv.data_ptr(),
                                      torch.cuda.current_stream().cuda_stream) == pkg.LSP_OK
    torch.cuda.synchronize()
    assert int(pi[0]) == int(np.argmax(P_only.cpu().numpy()))


def test_static_entry_point_allocates_nothing(lsp):
    """Device free memory is the same before and after a call (the first call on a device may load the module: warm up first),
    and the call can be captured into a CUDA graph and replayed -- a cudaMalloc or cudaFree under capture is an error."""
    import torch
    pkg, h = lsp
    w = workloads.c2()
    t, x = torch.from_numpy(w.t).cuda(), torch.from_numpy(w.x).cuda()
    P = torch.empty(w.Nf, dtype=torch.float32, device="cuda")
    pi = torch.zeros(1, dtype=torch.int32, device="cuda"); pv = torch.zeros(1, dtype=torch.float32, device="cuda")
    pkg.periodogram_static(t, x, w.f_min, w.df, w.Nf, out=P, peak_idx=pi, peak_val=pv)           # warm-up
    torch.cuda.synchronize()
    eager = P.clone()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(5):
        pkg.periodogram_static(t, x, w.f_min, w.df, w.Nf, out=P, peak_idx=pi, peak_val=pv)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(s):
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=s):
            pkg.periodogram_static(t, x, w.f_min, w.df, w.Nf, out=P, peak_idx=pi, peak_val=pv)
    for _ in range(2):
        P.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(P, eager)
    assert int(pi[0]) == int(torch.argmax(eager))


def test_static_entry_point_limits(lsp):
    """Beyond Nt = 16,384 or Nf = 262,144: LSP_ELIMIT and nothing written.  AT the limits the call runs, with the time splits cut
    to what the array holds, and agrees with the existing path."""
    import torch
    pkg, h = lsp
    assert (pkg.STATIC_MAX_NT, pkg.STATIC_MAX_NF, pkg.STATIC_SCRATCH_BYTES) == (16384, 262144, 8 << 20)
    rng = np.random.default_rng(12)
    Nt, Nf = pkg.STATIC_MAX_NT, pkg.STATIC_MAX_NF
    tt = np.sort(rng.uniform(0.0, 400.0, Nt + 1))
    xx = (rng.standard_normal(Nt + 1) + 0.3 * np.sin(2 * np.pi * 3.21 * tt)).astype(np.float32)
    t, x = torch.from_numpy(tt).cuda(), torch.from_numpy(xx).cuda()
    f_min, df = 1.0 / 400.0, (20.0 - 1.0 / 400.0) / (Nf - 1)
    P = torch.full((Nf + 1,), -1.0, dtype=torch.float32, device="cuda")
    for nt, nf in ((Nt + 1, 1000), (1000, Nf + 1)):
        with pytest.raises(pkg.LspError) as ei:
            pkg.periodogram_static(t[:nt].contiguous(), x[:nt].contiguous(), f_min, df, nf, out=P)
        assert ei.value.status == pkg.LSP_ELIMIT and "limits" in str(ei.value)
    torch.cuda.synchronize()
    assert float(P.min()) == -1.0 and float(P.max()) == -1.0
    with pytest.raises(pkg.LspError) as ei:
        pkg.periodogram_static(t[:1].contiguous(), x[:1].contiguous(), f_min, df, 10, out=P)
    assert ei.value.status == pkg.LSP_EINVAL
    t0, x0 = t[:Nt].contiguous(), x[:Nt].contiguous()
    Pe, pie, pve = _existing(pkg, h, t0, x0, f_min, df, Nf)
    Ps, pis, pvs = _static(pkg, t0, x0, f_min, df, Nf)
    assert np.max(np.abs(Ps - Pe)) <= TOL * float(Pe.max())
    assert pis == int(np.argmax(Ps))
    ks = np.unique(np.concatenate([np.arange(0, Nf, 4099), [pis, Nf - 1]])).astype(np.int64)
    ref = oracle.periodogram(tt[:Nt], xx[:Nt], f_min, df, Nf, ks=ks)
    assert np.max(np.abs(Ps[ks] - ref)) <= TOL * float(ref.max())
