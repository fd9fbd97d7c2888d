"""mdwf_nucleon_2pt_noalloc: the nucleon two-point contraction for callers that must
not allocate -- its per-warp partial sums live in a fixed file-scope device array instead of coming from
cudaMallocAsync (include/mdwf.h).  Checked against the existing path (mdwf_nucleon_2pt) on two calls in a row with
different inputs (the shared array keeps the previous call's contents, which must not leak into the next result), for
no change in free device memory across a call, and for a clear refusal beyond the array's size.

Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu

TOL = 1e-12          # the bound tests/test_gpu_meas.py uses for this contraction (fp64, fixed-order sums)


def rel(a, b):
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def crandn(shape, seed):
    g = torch.Generator().manual_seed(seed)
    return torch.complex(torch.randn(shape, generator=g, dtype=torch.float64), torch.randn(shape, generator=g, dtype=torch.float64))


def test_noalloc_matches_existing_path_on_two_calls_in_a_row():
    import paper_1810_01609_b200 as mdwf
    dims = (4, 6, 4, 8)
    T = dims[3]
    ctx = mdwf.Context(dims, 4, 1.3, 1.5, 0.5, 0.1)
    V4 = int(np.prod(dims))
    S = [crandn((12, V4, 4, 3), 9100 + i).cuda() for i in range(4)]
    g = [oracle.gamma(m) for m in range(4)]
    P_unpol = 0.5 * (np.eye(4) + g[3])
    P_pol = 0.25 * (np.eye(4) + g[3]) @ (np.eye(4) + 1j * g[0] @ g[1])
    calls = [((S[0], S[1], S[2]), P_unpol, 0), ((S[3], S[0], S[1]), P_pol, 3)]      # second call: other inputs, projector, t0
    want = [ctx.mdwf_nucleon_2pt(*s, P, t0=t0).cpu().numpy() for s, P, t0 in calls]
    assert rel(want[0], want[1]) > 0.1                      # the two calls really have different answers
    corr = torch.full((T, 2), float("nan"), dtype=torch.float64, device="cuda")      # caller-supplied output
    torch.cuda.synchronize()
    for k, (s, P, t0) in enumerate(calls):                  # back to back on one stream, same output buffer
        free0 = torch.cuda.mem_get_info()[0]
        got = ctx.mdwf_nucleon_2pt_noalloc(*s, P, corr, t0=t0)
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info()[0]
        got = got.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert rel(got, want[k]) <= TOL, (k, rel(got, want[k]))
        if k == 1:                                          # (the first call may still load the module lazily)
            assert free1 == free0, "device memory changed across a no-alloc call: %d -> %d" % (free0, free1)
    # and against the oracle's literal index sums, like the existing path's own test
    s, P, t0 = calls[1]
    exp = oracle.nucleon_2pt(dims, *[x.cpu().numpy() for x in s], P, t0=t0)
    assert rel(ctx.mdwf_nucleon_2pt_noalloc(*s, P, corr, t0=t0).cpu().numpy(), exp) <= TOL
    # repeating the first call after the second gives the first answer again
    s, P, t0 = calls[0]
    assert rel(ctx.mdwf_nucleon_2pt_noalloc(*s, P, corr, t0=t0).cpu().numpy(), want[0]) <= TOL


def test_noalloc_refuses_what_does_not_fit():
    import paper_1810_01609_b200 as mdwf
    from paper_1810_01609_b200.binding import lib
    cap = lib().mdwf_nucleon_2pt_noalloc_max_bytes()
    assert cap == 512 * 1024
    dims = (2, 2, 2, 6556)          # one block per timeslice: 10 * T doubles = 524480 bytes > 512 KiB
    ctx = mdwf.Context(dims, 1, 1.3, 1.5, 0.5, 0.1)
    V4 = int(np.prod(dims))
    S = crandn((12, V4, 4, 3), 9200).cuda()
    P = 0.5 * (np.eye(4) + oracle.gamma(3))
    corr = torch.full((dims[3], 2), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(mdwf.MdwfError) as e:
        ctx.mdwf_nucleon_2pt_noalloc(S, S, S, P, corr)
    assert "scratch" in str(e.value) and str(cap) in str(e.value)
    torch.cuda.synchronize()
    assert torch.all(corr == 7.0)                                        # nothing was written
    ref = ctx.mdwf_nucleon_2pt(S, S, S, P)                               # the allocating path still serves this size
    assert torch.all(torch.isfinite(torch.view_as_real(ref)))
