"""qmc_lattice_integrate_batch_static -- the entry that allocates nothing (workspace = a device array inside the library image).

Collected last on purpose (the suite runs with pytest -x).  Checks the new entry against the existing stream-ordered path
(qmc_lattice_integrate_batch with a caller-allocated workspace) on two calls in a row, within the tolerance of the parity tests
(1e-13 relative per shift mean, tests/test_gpu_parity.py); the two paths run the same kernels, so the bits agree as well.
"""
import numpy as np
import pytest

from paper_1811_11720_b200 import binding, synth

pytestmark = pytest.mark.gpu

REL_MEANS = 1e-13
K = synth.TRANSFORM_KOROBOV


def _problems():
    """one closed-form problem alone (travels in the kernel parameter), and a mixed batch with sectors (prepare kernel, tile queues)"""
    single = [synth.config(1, n_override=65521)[0]]
    batch = synth.config(3, n_override=8191, count_override=6) + [synth.config(0)[0], synth.config(2, n_override=4093)[0]]
    return single, batch


def _close(a, b):
    a, b = np.asarray(a), np.asarray(b)
    scale = np.maximum(np.abs(b), 1e-300)
    return np.all(np.abs(a - b) <= REL_MEANS * scale)


@pytest.mark.parametrize("which", [0, 1])
def test_static_entry_matches_the_workspace_path_twice_in_a_row(which):
    import torch
    probs = _problems()[which]
    ref = binding.DeviceBatch(probs)
    ref.integrate()
    sm_ref, means_ref, errs_ref = ref.results()
    assert np.all(np.isfinite(means_ref))
    stat = binding.DeviceBatch(probs)
    assert int(binding.lib().qmc_workspace_bytes(stat.count, stat.arr)) <= int(binding.lib().qmc_static_scratch_bytes())
    for call in range(2):
        stat.means.fill_(float("nan"))
        stat.errs.fill_(float("nan"))
        stat.shift_means.fill_(float("nan"))
        launches = stat.integrate_static()
        assert launches >= 2
        sm, means, errs = stat.results()
        for i in range(len(probs)):
            assert _close(sm[i], sm_ref[i]), (call, probs[i]["name"])
        nc = [binding.qmc_num_components(p["family"]) for p in probs]
        for i, c in enumerate(nc):
            assert _close(means[i, :c], means_ref[i, :c]) and _close(errs[i, :c], errs_ref[i, :c]), (call, probs[i]["name"])
            # the same kernels on the same tiles: bit identity, not just the tolerance
            assert sm[i].tobytes() == sm_ref[i].tobytes()
    torch.cuda.synchronize()


def test_static_entry_after_another_batch_used_the_scratch():
    """the array keeps the last call's contents: a small problem right after a large batch must not see them"""
    single, batch = _problems()
    big = binding.DeviceBatch(batch)
    big.integrate_static()
    big.results()
    ref = binding.DeviceBatch(single)
    ref.integrate()
    sm_ref, _, _ = ref.results()
    small = binding.DeviceBatch(single)
    small.integrate_static()
    sm, _, _ = small.results()
    assert sm[0].tobytes() == sm_ref[0].tobytes()


def test_static_entry_rejects_what_does_not_fit():
    """a batch whose workspace exceeds the static array is refused before anything is launched, with a text that says why"""
    L = binding.lib()
    limit = int(L.qmc_static_scratch_bytes())
    assert limit == 4 * 1024 * 1024
    p = synth.config(0)[0]
    many = [dict(p, name=f"p{i}") for i in range(2000)]
    batch = binding.DeviceBatch(many)
    need = int(L.qmc_workspace_bytes(batch.count, batch.arr))
    assert need > limit
    with pytest.raises(binding.QmcError) as e:
        batch.integrate_static()
    assert e.value.status == -11                                 # QMC_ERR_WORKSPACE
    text = L.qmc_last_cuda_error().decode()
    assert str(need) in text and str(limit) in text
    batch.integrate()                                            # the workspace path still serves it
    _, means, _ = batch.results()
    assert np.all(np.isfinite(means[:, 0]))
    # argument checks come first
    assert L.qmc_lattice_integrate_batch_static(0, batch.arr, None, None, None, None) == -3
    assert L.qmc_lattice_integrate_batch_static(1, None, None, None, None, None) == -1
