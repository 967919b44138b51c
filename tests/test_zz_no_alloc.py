"""gvqe_argmax_noalloc (include/gvqe.h): the read-out sweep of gvqe_argmax with its per-block candidates in
a file-scope device array, for callers that may not allocate device memory.  Checked against the existing path
(gvqe_argmax on the same amplitudes: the two run the same kernels over the same partition, so index and probability
must be equal, not just close) on two calls in a row that share the scratch array -- the second over a smaller state,
so that the array still holds entries of the first call that the second must not read.

Named test_zz_* so that pytest collects it last: a failure here hides no other test under `pytest -x`."""
import numpy as np
import pytest

import paper_2607_02749_b200 as gv
from workload import make_workload


def _existing_path(w, prec, slot):
    """gvqe_argmax on the state of row `slot`, and that state (host copy of the kernel's own amplitudes)."""
    g = gv.Gvqe(w.n, layout=dict(n_layers=w.D, entangler=w.entangler, topology=w.topology, final_rot=w.final_rot), precision=prec)
    g.set_hamiltonian(w.paulis, w.coeffs)
    g.alloc_workspace(2)
    g.energy_batch(w.params)
    x, p = g.argmax(slot)
    psi = g.get_state(slot)
    g.close()
    return x, p, psi


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["c64", "c128"])
def test_argmax_noalloc_matches_argmax_on_two_calls_in_a_row(prec):
    import torch

    dev = torch.device("cuda:0")
    cdt = torch.complex64 if prec == "c64" else torch.complex128
    cases = [make_workload(4, n=21, M=30, D=2, batch=2), make_workload(3, n=12, M=30, D=2, batch=2)]   # 2^21, then 2^12 amplitudes
    refs = [_existing_path(w, prec, slot=1) for w in cases]
    states = [torch.from_numpy(np.ascontiguousarray(psi)).to(dev).to(cdt) for (_, _, psi) in refs]
    results = [torch.zeros(2, dtype=torch.int64, device=dev) for _ in cases]   # 16 bytes each: {float64 prob, uint64 x}
    stream = torch.cuda.current_stream().cuda_stream
    before = torch.cuda.memory_allocated()
    for st, res in zip(states, results):                      # back to back on one stream, no synchronisation between them
        gv.argmax_noalloc(st.data_ptr(), st.numel(), prec, res.data_ptr(), stream)
    assert torch.cuda.memory_allocated() == before
    torch.cuda.synchronize()
    for (x_ref, p_ref, psi), res in zip(refs, results):
        out = res.cpu().numpy()
        x, p = int(out.view(np.uint64)[1]), float(out.view(np.float64)[0])
        assert x == x_ref and p == p_ref
        pk = psi.real * psi.real + psi.imag * psi.imag        # the kernel's decision rule on its own amplitudes, ties to the lowest x
        assert x == int(np.argmax(pk)) and p == float(pk[x])
    # the same call again on the first state: whatever the calls above left in the scratch array changes nothing
    gv.argmax_noalloc(states[0].data_ptr(), states[0].numel(), prec, results[1].data_ptr(), stream)
    torch.cuda.synchronize()
    out = results[1].cpu().numpy()
    assert int(out.view(np.uint64)[1]) == refs[0][0] and float(out.view(np.float64)[0]) == refs[0][1]


def test_argmax_noalloc_rejects_bad_sizes():
    """Argument checks come before any CUDA call (host only): sizes beyond the stated maximum, empty states, bad pointers."""
    for args, word in (((256, gv.NOALLOC_MAX_AMPLITUDES + 1, "c64", 256), "exceed the maximum"), ((256, 0, "c128", 256), "is 0"),
                       ((0, 16, "c64", 256), "NULL"), ((256, 16, "c64", 0), "NULL"), ((264, 16, "c64", 256), "aligned")):
        with pytest.raises(gv.GvqeError) as e:
            gv.argmax_noalloc(*args)
        assert e.value.status == gv.GVQE_ERR_INVALID_ARG and word in str(e.value)
