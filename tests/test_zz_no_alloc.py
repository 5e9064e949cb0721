"""fcg_break_step_static (include/fcg.h): the break step for callers that may not allocate -- no handle, no workspace, its scratch
in a static device array inside libfcg.so.  Checked against the existing path (fcg_break_step on a handle) on the same inputs,
two calls in a row (the second call finds the static array as the first one left it, and k with the first winner removed):
index, ratio and the updated k must agree BIT FOR BIT, the bar tests/test_gpu_parity.py::test_break_step_matches_oracle sets for
this integer / IEEE-divide work.  This file is named to be collected last (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from paper_1305_3625_b200 import inputs

pytestmark = pytest.mark.gpu
TDT = {np.float64: torch.float64, np.float32: torch.float32}


@pytest.fixture(scope="module")
def B():
    from paper_1305_3625_b200 import binding
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    binding.lib()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def case(L, dt, seed):
    rng = np.random.default_rng(seed)
    N = L * L
    k = (rng.random(N) + 0.5).astype(dt); k[rng.random(N) < 0.3] = 0
    u = rng.standard_normal(N).astype(dt); t = rng.random(N).astype(dt)
    u[5] = u[3]; t[5] = t[3]; k[5] = k[3] = 1.0                       # an exact tie somewhere: lowest index wins
    return k, u, t


@pytest.mark.parametrize("L,dt", [(64, np.float64), (512, np.float64), (512, np.float32), (2048, np.float32), (2048, np.float64)])
def test_break_step_static_matches_handle_path(B, L, dt):
    k, u, t = case(L, dt, 23 + L)
    h = B.Fcg(L, TDT[dt])
    k_ref, k_new, ud, td = dev(k), dev(k), dev(u), dev(t)
    res = torch.zeros(3, dtype=torch.int64, device="cuda")
    for call in range(2):                                             # two calls in a row on the shared static scratch
        idx, ratio, st = h.fcg_break_step(k_ref, ud, td)
        B.fcg_break_step_static(k_new, ud, td, res)
        idx2, ratio2, st2 = B.break_result(res)
        assert (idx2, ratio2, st2) == (idx, ratio, st), (call, idx2, idx, ratio2, ratio)
        assert idx >= 0 and torch.equal(k_new, k_ref) and float(k_new.view(-1)[idx]) == 0.0
    h.close()


def test_break_step_static_rules_and_no_candidate(B):
    """S13 on the allocation-free path: t = 0 gives +inf and wins, 0/0 = NaN is skipped, nothing left -> index -1, FCG_NO_CANDIDATE;
    a ragged n (not a multiple of the vector width, not a square) against a plain numpy evaluation of the rule."""
    k = np.zeros(256); u = np.zeros(256); t = np.ones(256)
    k[200] = 1.0; u[200] = 2.0; t[200] = 0.0; k[100] = 1.0; t[100] = 0.0
    kd, res = dev(k), torch.zeros(3, dtype=torch.int64, device="cuda")
    B.fcg_break_step_static(kd, dev(u), dev(t), res)
    idx, ratio, st = B.break_result(res)
    assert idx == 200 and np.isinf(ratio) and st == 0
    B.fcg_break_step_static(kd, dev(u), dev(t), res)
    assert B.break_result(res)[0] == -1 and B.break_result(res)[2] == B.FCG_NO_CANDIDATE
    rng = np.random.default_rng(5)
    n = 100003
    buf = [torch.zeros(n + 4, dtype=torch.float64, device="cuda")[:n] for _ in range(3)]       # 16-byte aligned bases, ragged length
    kh = rng.random(n) + 0.5; kh[rng.random(n) < 0.5] = 0; uh = rng.standard_normal(n); th = rng.random(n)
    for b, a in zip(buf, (kh, uh, th)):
        b.copy_(torch.from_numpy(a))
    B.fcg_break_step_static(buf[0], buf[1], buf[2], res)
    idx, ratio, st = B.break_result(res)
    r = np.where(kh > 0, (kh * uh) / th, -np.inf)
    assert idx == int(np.argmax(r)) and ratio == r[idx] and st == 0


def test_break_step_static_limits_and_no_allocation(B):
    """Sizes beyond the stated maximum and misaligned pointers are refused with a message; a call allocates no device memory
    (free memory as the driver reports it is unchanged) and is legal under stream capture, where cudaMalloc is not."""
    lib = B.lib()
    x = torch.ones(1024, dtype=torch.float64, device="cuda")
    res = torch.zeros(3, dtype=torch.int64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    rc = lib.fcg_break_step_static(B.FCG_F64, B.FCG_BREAK_STATIC_MAX_N + 1, x.data_ptr(), x.data_ptr(), x.data_ptr(), res.data_ptr(), st)
    assert rc == B.FCG_UNSUPPORTED and b"FCG_BREAK_STATIC_MAX_N" in lib.fcg_static_last_error()
    rc = lib.fcg_break_step_static(B.FCG_F64, 512, x.data_ptr() + 8, x.data_ptr(), x.data_ptr(), res.data_ptr(), st)
    assert rc == B.FCG_INVALID_ARG and b"aligned" in lib.fcg_static_last_error()
    assert lib.fcg_break_step_static(B.FCG_F64, 0, x.data_ptr(), x.data_ptr(), x.data_ptr(), res.data_ptr(), st) == B.FCG_INVALID_ARG
    k, u, t = (dev(a) for a in case(512, np.float64, 3))
    B.fcg_break_step_static(k.clone(), u, t, res)                     # first call on this device: symbol address looked up
    torch.cuda.synchronize()
    k1, k2 = k.clone(), k.clone()
    free0 = torch.cuda.mem_get_info()[0]
    B.fcg_break_step_static(k1, u, t, res)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    want = B.break_result(res)
    g = torch.cuda.CUDAGraph()
    res2 = torch.zeros(3, dtype=torch.int64, device="cuda")
    with torch.cuda.graph(g):                                         # capture error mode "global": an allocation here would raise
        B.fcg_break_step_static(k2, u, t, res2)
    g.replay()
    torch.cuda.synchronize()
    assert B.break_result(res2) == want and torch.equal(k1, k2)
