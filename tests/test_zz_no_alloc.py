"""pt_gimenez_interp_static (include/pt.h): the Giménez z-interpolation with its work area in a fixed array of the library,
for callers that cannot allocate device memory.  Checked against the existing path (pt_gimenez_interp, caller-owned work
area) on two calls in a row of different shapes — the second must not be disturbed by what the first left in the array.
Collected last on purpose (the file name): the suite runs with pytest -x."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-12        # the gate of the interpolated Giménez path in test_gpu_parity.py


def _population(n_pv, n_pb, n_ldc, seed):
    rng = np.random.default_rng(seed)
    P, a = rng.uniform(1, 10, n_pv), rng.uniform(4, 20, n_pv)
    e = np.where(rng.uniform(size=n_pv) < 0.5, 0.0, rng.uniform(0, 0.5, n_pv))
    wv = rng.uniform(0, 2 * math.pi, n_pv)
    inc = np.arccos(np.clip(rng.uniform(0, 0.9, n_pv) * (1 + e * np.sin(wv)) / (a * (1 - e * e)), -1, 1))
    k = rng.uniform(0.02, 0.3, n_pv)
    u = rng.uniform(-0.1, 0.5, (n_pv, n_pb * n_ldc)) / n_ldc
    params = np.concatenate([np.stack([P * rng.uniform(0, 1, n_pv), P, a, inc, e, wv, k], 1), u], 1)
    t14 = P / (math.pi * a)
    return params, t14, rng


def _dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def test_gimenez_interp_static_matches_caller_owned_work_area():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1504_07433_b200 as pt
    from paper_1504_07433_b200 import binding
    L = binding.lib()
    assert L.pt_build_arch() == 100
    cap = pt.pt_gimenez_static_work_doubles()
    assert cap == 1 << 19

    # two calls in a row, the second with a different (smaller) table layout, one bad row and supersampling
    cases = [dict(n_pv=40, n_pb=2, n_ldc=3, n_j=30, n_in=200, n_out=300, n_t=900, n_ss=1, t_exp=0.0, seed=11, bad=None),
             dict(n_pv=7, n_pb=1, n_ldc=2, n_j=20, n_in=33, n_out=47, n_t=257, n_ss=3, t_exp=0.004, seed=12, bad=2)]
    prepared = []
    for c in cases:
        params, t14, rng = _population(c["n_pv"], c["n_pb"], c["n_ldc"], c["seed"])
        t = params[:, 0][:, None] + rng.uniform(-1.2, 1.2, (c["n_pv"], c["n_t"])) * t14[:, None]
        if c["bad"] is not None:
            params[c["bad"], 1] = -1.0
        coef = pt.GimenezCoef(c["n_ldc"], c["n_j"])
        ref, _ = pt.pt_gimenez_interp(coef, c["n_in"], c["n_out"], _dev(t), _dev(params), c["n_pb"], c["n_ss"], c["t_exp"])
        out = torch.full((c["n_pv"], c["n_pb"], c["n_t"]), -7.0, dtype=torch.float64, device="cuda")
        st = torch.zeros(2, dtype=torch.int32, device="cuda")
        prepared.append((c, coef, _dev(t), _dev(params), ref, out, st))
    torch.cuda.synchronize()

    for i, (c, coef, t, params, ref, out, st) in enumerate(prepared):
        free0 = torch.cuda.mem_get_info()[0]
        pt.pt_gimenez_interp_static(coef, c["n_in"], c["n_out"], t, params, out, c["n_pb"], c["n_ss"], c["t_exp"], status=st)
        torch.cuda.synchronize()
        if i > 0:       # (the first call of a process may load the module's code)
            assert torch.cuda.mem_get_info()[0] == free0, "the call changed the amount of free device memory"
        f, r = out.cpu().numpy(), ref.cpu().numpy()
        assert np.array_equal(np.isnan(f), np.isnan(r))
        ok = ~np.isnan(r)
        assert np.abs(f[ok] - r[ok]).max() <= TOL
        assert (r[ok] < 1.0).mean() > 0.2 and not np.any(f[ok] == -7.0)
        if c["bad"] is not None:
            assert np.all(np.isnan(f[c["bad"]])) and st.cpu().tolist() == [pt.PT_ST_BAD_PARAM, 1]
        else:
            assert st.cpu().tolist() == [0, 0]

    # the first case again after the second: same result as before (the array is simply overwritten)
    c, coef, t, params, ref, out, st = prepared[0]
    out.fill_(-7.0)
    pt.pt_gimenez_interp_static(coef, c["n_in"], c["n_out"], t, params, out, c["n_pb"], c["n_ss"], c["t_exp"])
    torch.cuda.synchronize()
    assert np.abs(out.cpu().numpy() - ref.cpu().numpy()).max() <= TOL

    # beyond the maximum: a clear error, nothing enqueued, the output untouched
    n_ldc, n_in, n_out = 3, 200, 300
    n_pv_max = cap // ((n_ldc + 1) * (n_in + n_out))
    big = np.tile(prepared[0][3].cpu().numpy()[:1], (n_pv_max + 1, 1))
    tt = prepared[0][2][0].contiguous()
    o = torch.full((n_pv_max + 1, 2, tt.numel()), -7.0, dtype=torch.float64, device="cuda")
    coef = prepared[0][1]
    n0 = pt.pt_launch_count()
    with pytest.raises(pt.PtError, match="PT_ERR_SIZE"):
        pt.pt_gimenez_interp_static(coef, n_in, n_out, tt, _dev(big), o, 2)
    assert pt.pt_launch_count() == n0
    torch.cuda.synchronize()
    assert bool((o == -7.0).all())
    # exactly at the maximum it runs
    o2 = pt.pt_gimenez_interp_static(coef, n_in, n_out, tt, _dev(big[:n_pv_max]), o[:n_pv_max].contiguous(), 2)
    ref2, _ = pt.pt_gimenez_interp(coef, n_in, n_out, tt, _dev(big[:n_pv_max]), 2)
    assert np.abs(o2.cpu().numpy() - ref2.cpu().numpy()).max() <= TOL
    # the other argument errors come back as from pt_gimenez_interp
    p1 = _dev(big[:1])
    assert L.pt_gimenez_interp_static(None, 3, 30, 20, 20, tt.data_ptr(), tt.numel(), 0, p1.data_ptr(), 1, 2, 1, 0.0,
                                      o.data_ptr(), None, None) == binding.PT_ERR_NULL
    assert L.pt_gimenez_interp_static(coef.data.data_ptr(), 3, 30, 1, 20, tt.data_ptr(), tt.numel(), 0, p1.data_ptr(), 1, 2, 1,
                                      0.0, o.data_ptr(), None, None) == binding.PT_ERR_SIZE
    assert L.pt_gimenez_interp_static(coef.data.data_ptr(), 3, 30, 1 << 30, 1 << 30, tt.data_ptr(), tt.numel(), 0, p1.data_ptr(),
                                      1, 2, 1, 0.0, o.data_ptr(), None, None) == binding.PT_ERR_SIZE
