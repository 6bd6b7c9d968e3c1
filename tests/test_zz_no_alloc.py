"""gwmf_power_table_static -- the entry point for callers that cannot allocate device memory.

Most of the library works out of a workspace the caller hands to gwmf_create.  A caller that must not call cudaMalloc
when its PSD changes (an online search whose running filters an allocation would stall, a process whose GPU memory a
caching allocator already owns, a plug-in that may only touch the buffers it is given) has no workspace to hand over,
so this one entry point keeps its scratch in a static array inside the library image and allocates nothing.

The GPU test checks its output against the existing workspace path (gwmf_load_segment -> gwmf_sigma / gwmf_band_edges,
which are derived from the same table) on two calls in a row with different PSDs and then a third with the first PSD
again: the scratch is shared by all calls and keeps the last call's contents, so a call that relied on stale
contents, or failed to reset the status word, would show up in the second or third call.

The file sorts last on purpose (pytest -x stops at the first failure and would hide every test after it).  It passes
both alone in a fresh process (then its first call is the one that resolves the static array's device address) and
after the other GPU tests.
"""
import ctypes

import numpy as np
import pytest

import workloads as inputs

N = 1 << 20
P = 16
MASSES = [(1.0, 1.0), (1.4, 1.4), (2.0, 1.2), (3.0, 1.2), (5.0, 4.0), (8.0, 6.0), (12.0, 9.0), (20.0, 15.0),
          (1.0, 3.0), (10.0, 1.4), (30.0, 30.0), (45.0, 40.0)]


def _line_psd(n):
    """Eq. 2 with a strong line between 95 and 165 Hz: moves every band edge of every template."""
    Sn = inputs.psd_array(n).copy()
    df = inputs.FS / n
    Sn[int(95.0 / df):int(165.0 / df)] *= 1e4
    return Sn


def _from_table(Cj, k_high, p, n):
    """sigma and band edges from the power table, by the definitions include/gwmf.h states (Eq. 4)."""
    df = inputs.FS / n
    k_low = int(np.ceil(inputs.F_LOW / df))
    sig = np.empty(len(k_high))
    edges = np.empty((len(k_high), p + 1), dtype=np.int64)
    for t, kh in enumerate(k_high):
        total = Cj[kh - 1]
        sig[t] = np.sqrt(4.0 * df * total)
        edges[t, 0], edges[t, p] = k_low, kh
        for l in range(1, p):
            target = (float(l) / float(p)) * total
            edges[t, l] = k_low + int(np.searchsorted(Cj[k_low:kh], target, side="left")) + 1
    return sig, edges


@pytest.mark.gpu
def test_static_power_table_matches_the_workspace_path_on_consecutive_calls():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_0906_4175_b200 import gwmf
    psds = [inputs.psd_array(N), _line_psd(N), inputs.psd_array(N)]
    s = np.zeros(N, dtype=np.float32)                      # the table does not depend on the segment
    f = gwmf.Filter(N, P, 4096, len(MASSES), batch=2)
    f.make_bank(MASSES)
    out = torch.empty(N // 2, dtype=torch.float64, device="cuda:0")    # the caller's output buffer, reused by every call
    tables = []
    for i, Sn in enumerate(psds):
        # existing path: the table inside the context's workspace, seen through sigma and the band edges
        f.load_segment(s, Sn)
        sig_ws, edges_ws = f.sigma(), f.band_edges().astype(np.int64)
        # new entry point: same PSD, device-resident input, caller's output buffer, nothing allocated
        d_sn = torch.from_numpy(Sn).to("cuda:0")
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]         # the driver's count: sees a cudaMalloc made by anybody
        got = gwmf.power_table_static(d_sn, N, out=out)
        assert got is out
        if i > 0:                                          # (the first launch of a kernel may make the driver load its code)
            assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
        Cj = out.cpu().numpy()
        tables.append(Cj.copy())
        assert np.all(np.diff(Cj) >= 0.0) and Cj[0] == 0.0
        sig, edges = _from_table(Cj, edges_ws[:, P], P, N)
        assert np.array_equal(edges, edges_ws), f"call {i}: band edges differ from the workspace path"
        # tests/parity.py compares sigma to 1e-5 relative; the two tables are summed in the same order, so ask for far more
        assert np.all(np.abs(sig - sig_ws) <= 1e-13 * sig_ws), f"call {i}: sigma {sig} vs {sig_ws}"
    assert not np.array_equal(tables[0], tables[1])        # the second PSD really was a different problem
    assert tables[0].tobytes() == tables[2].tobytes()      # nothing of call 2 survives into call 3

    # a bad PSD is reported, and the status word it raised does not leak into the next call
    bad = torch.from_numpy(psds[0].copy()).to("cuda:0")
    bad[N // 8] = -1.0
    with pytest.raises(gwmf.GwmfError) as ei:
        gwmf.power_table_static(bad, N, out=out)
    assert ei.value.status == gwmf.E_ARG and "S_n" in str(ei.value)
    gwmf.power_table_static(torch.from_numpy(psds[0]).to("cuda:0"), N, out=out)
    assert out.cpu().numpy().tobytes() == tables[0].tobytes()

    # other sizes, smallest included: same check against a context of that size
    for n in (1 << 14, 1 << 17):
        Sn = inputs.psd_array(n)
        g = gwmf.Filter(n, 4, 4096, 2)
        g.make_bank([(8.0, 8.0), (1.4, 1.4)])
        g.load_segment(np.zeros(n, dtype=np.float32), Sn)
        e_ws = g.band_edges().astype(np.int64)
        Cj = gwmf.power_table_static(torch.from_numpy(Sn).to("cuda:0"), n).cpu().numpy()
        sig, edges = _from_table(Cj, e_ws[:, 4], 4, n)
        assert np.array_equal(edges, e_ws) and np.all(np.abs(sig - g.sigma()) <= 1e-13 * sig)
        g.close()
    f.close()


def test_static_power_table_rejects_sizes_beyond_its_scratch_without_a_gpu():
    """Argument checks come before any CUDA call, so they can be exercised on a CPU-only box: a segment longer than
    GWMF_STATIC_MAX_N is refused with GWMF_E_CAPACITY and a message that says why and what to use instead."""
    from paper_0906_4175_b200 import build, gwmf
    build.build()
    L = gwmf.load_library()
    err = ctypes.create_string_buffer(256)
    dummy = ctypes.c_void_p(256)                           # never dereferenced: the size check fails first
    rc = L.gwmf_power_table_static(dummy, dummy, gwmf.STATIC_MAX_N * 2, 4096.0, 40.0, None, err, len(err))
    assert rc == gwmf.E_CAPACITY
    text = err.value.decode()
    assert str(gwmf.STATIC_MAX_N) in text and "workspace" in text, text
    assert L.gwmf_power_table_static(dummy, dummy, 3 << 13, 4096.0, 40.0, None, err, len(err)) == gwmf.E_ARG
    assert L.gwmf_power_table_static(dummy, dummy, 1 << 13, 4096.0, 40.0, None, err, len(err)) == gwmf.E_ARG
    assert L.gwmf_power_table_static(None, dummy, 1 << 20, 4096.0, 40.0, None, err, len(err)) == gwmf.E_ARG
    assert L.gwmf_power_table_static(dummy, dummy, 1 << 20, 4096.0, 4096.0, None, None, 0) == gwmf.E_ARG
