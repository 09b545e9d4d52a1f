"""tpc_fit_tracks_noalloc: the three-iteration fit with its scratch in a static array inside the library
(include/tpc_track.h).  Collected last on purpose (the file name): the suite runs with pytest -x.

The new entry point runs the same fit as tpc_fit_tracks on the same inputs: its output must equal the existing
path's bit for bit in the deterministic build and within the fast-mode tolerance in the fast build; checked on
calls in a row on frames of different sizes, which share the one array (what a call leaves behind must not
reach the next one).
"""
import numpy as np
import pytest

from paper_2601_20569_b200 import datagen as dg

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_20569_b200 import binding
    binding.load_library()
    return binding


class Case:
    """A frame carried through the EXISTING path (track, refit, merge, fit with a caller workspace); keeps the
    device buffers the no-allocation call takes as inputs."""

    def __init__(self, B, clusters, flags):
        import torch
        self.B, self.torch, self.flags = B, torch, flags
        self.trk = B.SectorTracker()
        self.d_clusters = self.trk.upload(clusters)
        self.n_clusters = len(clusters)
        self.trk.track(self.d_clusters, flags=flags)
        self.trk.counts()
        self.trk.refit()
        self.trk.merge(fetch=False)
        self.fit, self.chi2, self.rejected = self.trk.fit()               # the existing path's result
        rc, self.d_refit = B.tpc_get_refit(self.trk.ctx)
        assert rc == B.TPC_OK
        rc, self.mv = B.tpc_get_merged(self.trk.ctx)
        assert rc == B.TPC_OK
        nm, ni = int(self.mv.n_merged), int(self.mv.n_cluster_ids)
        assert nm == len(self.fit) > 0 and ni == len(self.chi2) <= B.TPC_FIT_NOALLOC_MAX_IDS
        # the caller's outputs, filled with a pattern the call must overwrite
        self.o_fit = torch.full((nm * B.TRACK_FIT3_DTYPE.itemsize,), 0xA5, dtype=torch.uint8, device="cuda")
        self.o_chi2 = torch.full((ni,), -7.0, dtype=torch.float32, device="cuda")
        self.o_rej = torch.full((ni,), 0xA5, dtype=torch.uint8, device="cuda")

    def call(self, n_cluster_ids=None, fit_out=None):
        B, mv = self.B, self.mv
        st = self.torch.cuda.current_stream().cuda_stream
        return B.tpc_fit_tracks_noalloc(
            self.trk.ctx, None, self.d_clusters.data_ptr(), self.n_clusters, self.d_refit, int(mv.n_tracks), mv.d_merged,
            int(mv.n_merged), mv.d_seg_index, mv.d_cluster_ids, int(mv.n_cluster_ids) if n_cluster_ids is None else n_cluster_ids,
            self.o_fit.data_ptr() if fit_out is None else fit_out, self.o_chi2.data_ptr(), self.o_rej.data_ptr(),
            self.flags & B.TPC_DETERMINISTIC, st)

    def check(self):
        """Deterministic build: bit for bit.  Fast build: the workspace path reads a compact copy of the clusters
        and is another instantiation of the kernel than the one this entry point runs (it gathers from the
        frame), so the two may differ in the last bits: the fast-mode tolerance of the other tests (1e-3
        relative on parameters and chi2, decisions at a cut may flip for a handful of clusters)."""
        B = self.B
        self.torch.cuda.synchronize()
        fit = self.o_fit.cpu().numpy().view(B.TRACK_FIT3_DTYPE)
        chi2, rej = self.o_chi2.cpu().numpy(), self.o_rej.cpu().numpy()
        if self.flags & B.TPC_DETERMINISTIC:
            assert fit.tobytes() == self.fit.tobytes()
            assert chi2.tobytes() == self.chi2.tobytes()
            assert (rej == self.rejected).all()
            return
        assert (rej != self.rejected).sum() <= 1e-4 * len(rej) + 2
        assert np.allclose(chi2, self.chi2, rtol=1e-3, atol=1e-3)
        same = (fit["flags"] == self.fit["flags"]) & (fit["n_used"] == self.fit["n_used"])
        assert (~same).sum() <= 1e-3 * len(fit) + 2
        ok = same & (fit["flags"] == 0)
        scale = np.array([0.1, 0.1, 0.01, 0.01, 0.1], dtype=np.float64)
        a, b = fit["p"][ok].astype(np.float64), self.fit["p"][ok].astype(np.float64)
        bad = (np.abs(a - b) > 1e-3 * np.maximum(np.abs(b), scale)).any(axis=1)
        assert bad.sum() <= 5e-4 * ok.sum() + 2, int(bad.sum())
        assert np.allclose(fit["chi2"][ok], self.fit["chi2"][ok], rtol=2e-3, atol=1e-2)

    def scribble(self):
        self.o_fit.fill_(0x5A); self.o_chi2.fill_(-3.0); self.o_rej.fill_(0x5A)

    def close(self):
        self.trk.close()


@pytest.mark.parametrize("flags", [1, 0], ids=["det", "fast"])
def test_fit_without_allocation_equals_the_workspace_path(B, flags):
    import torch
    big, _, _ = dg.generate(dg.preset("C2", tracks_per_event=2000, seed=31))      # 36 sectors, ~2.8e5 clusters
    small, _, _ = dg.generate(dg.preset("C1"))                                     # one sector, ~1e4 clusters
    a, b = Case(B, big, flags), Case(B, small, flags)
    try:
        assert int(a.mv.n_cluster_ids) > 4 * int(b.mv.n_cluster_ids)
        assert (a.rejected != 0).any() and (a.fit["flags"] == 0).sum() > 0.9 * len(a.fit)
        assert a.call() == B.TPC_OK                   # (first use also loads the kernels of this entry point)
        a.check()
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        # calls in a row on the one shared array: large frame, small frame, large frame again, twice
        for case in (a, b, a, a, b):
            case.scribble()
            assert case.call() == B.TPC_OK
            case.check()
        # two calls enqueued back to back on one stream, checked afterwards
        a.scribble(); b.scribble()
        assert a.call() == B.TPC_OK and b.call() == B.TPC_OK
        a.check(); b.check()
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0   # no device memory was taken or given back by the calls
        # beyond the fixed maximum: refused with its own code and a text, nothing written
        a.scribble()
        assert a.call(n_cluster_ids=B.TPC_FIT_NOALLOC_MAX_IDS + 1) == B.TPC_E_LIMIT
        assert "TPC_FIT_NOALLOC_MAX_IDS" in B.tpc_last_cuda_error(a.trk.ctx)
        assert b"maximum" in B.load_library().tpc_strerror(B.TPC_E_LIMIT)
        torch.cuda.synchronize()
        assert (a.o_rej.cpu().numpy() == 0x5A).all()
        # null output, misaligned output
        assert a.call(fit_out=0) == B.TPC_E_ARG
        assert a.call(fit_out=a.o_fit.data_ptr() + 1) == B.TPC_E_ARG
        # the context's own state is untouched: its fit result is still there
        rc, fv = B.tpc_get_fit(a.trk.ctx)
        assert rc == B.TPC_OK and int(fv.n_merged) == len(a.fit)
    finally:
        a.close(); b.close()
