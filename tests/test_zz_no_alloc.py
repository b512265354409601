"""efm_beam_threshold_static(): the beam threshold for callers that cannot allocate device memory.

Some users of this library do not own the GPU they run on: their code is a step inside another program's GPU process
(a plug-in, a serving engine, a job under a hard memory cap) whose allocator holds all of HBM, or it sits in a loop where
cudaMalloc / cudaFree are banned because they can stall the device.  They can pass keys and a result slot, but no scratch.
efm_beam_threshold_static() keeps its scratch in an array compiled into the library (at most 2^20 keys per call).  The
GPU test below checks it, on consecutive calls that share that array, against

  * the existing path: efm_beam_threshold(), i.e. the launcher and kernels efm_enumerate() uses, scratch from the caller;
  * the definition: the key at sorted position cap among the selectable keys, by numpy's sort.

Integer work: the comparison is bit-exact, like every other parity test here.

This file is named test_zz_* so that pytest collects it last: with `-x` a failure here hides nothing behind it.  It must
pass alone in a fresh process (the first call then performs the per-device set-up) and after all other tests.
"""
import numpy as np
import pytest

import paper_1804_02867_b200 as efm

KEY_DONE = np.uint64(0xFFFFFFFFFFFFFFFE)       # balanced child: outside the ranking
KEY_SENTINEL = np.uint64(0xFFFFFFFFFFFFFFFF)   # unused slot / "keep everything"


def level_keys(n: int, seed: int, n_unb_max: int = 12, dup_every: int = 0) -> np.ndarray:
    """Key slots shaped like one level of the traversal: top byte = number of unbalanced metabolites (small, skewed to low
    values), 56 hash bits below, some balanced children and unused slots in between.  dup_every > 0 plants runs of equal keys."""
    rng = np.random.default_rng(seed)
    n_unb = np.minimum(rng.geometric(0.35, size=n), n_unb_max).astype(np.uint64)
    keys = (n_unb << np.uint64(56)) | (rng.integers(0, 1 << 56, size=n, dtype=np.uint64))
    if dup_every:
        keys[::dup_every] = keys[0]
    special = rng.random(n)
    keys[special < 0.05] = KEY_DONE
    keys[special > 0.97] = KEY_SENTINEL
    return keys


def threshold_by_definition(keys: np.ndarray, cap: int) -> int:
    live = np.sort(keys[keys < KEY_DONE])
    return int(live[cap]) if live.size > cap else int(KEY_SENTINEL)


def test_size_limit_is_refused_before_any_cuda_call():
    # no GPU needed: the limit is checked first, so a box without CUDA reports it the same way
    with pytest.raises(efm.EfmError) as ei:
        efm.beam_threshold_static(256, efm.STATIC_SELECT_MAX_KEYS + 1, 10, 512)
    assert ei.value.code == efm.EFM_E_CAPACITY
    assert "EFM_STATIC_SELECT_MAX_KEYS" in str(ei.value) and str(efm.STATIC_SELECT_MAX_KEYS) in str(ei.value)
    for bad in (dict(n=-1, cap=10, out=512), dict(n=10, cap=0, out=512), dict(n=10, cap=10, out=0)):
        with pytest.raises(efm.EfmError) as ei:
            efm.beam_threshold_static(256, bad["n"], bad["cap"], bad["out"])
        assert ei.value.code == efm.EFM_E_INVAL


@pytest.mark.gpu
def test_static_scratch_matches_existing_path_on_consecutive_calls():
    import torch
    dev = torch.device("cuda:0")

    # (n, cap, seed, dup_every); calls follow one another on one stream and share the built-in array:
    # a large call, a smaller one (stale compact keys of the first lie behind its own), ties at the threshold,
    # a beam that does not bind, the limit itself, a single tile, and the first case again
    cases = [(300_001, 65_536, 1, 0), (70_003, 1_000, 2, 0), (150_000, 40_000, 3, 3), (5_000, 5_000, 4, 0),
             (efm.STATIC_SELECT_MAX_KEYS, 262_144, 5, 0), (77, 5, 6, 0), (300_001, 65_536, 1, 0)]
    inputs = []
    for n, cap, seed, dup in cases:
        k = level_keys(n, seed, dup_every=dup)
        inputs.append((k, torch.from_numpy(k.view(np.int64)).to(dev)))
    # every buffer the calls need exists before the first call; the new entry point itself is given nothing but these
    out_static = torch.zeros(len(cases), dtype=torch.int64, device=dev)
    out_exist = torch.zeros(len(cases), dtype=torch.int64, device=dev)
    scratch = torch.empty(efm.beam_threshold_scratch_bytes(efm.STATIC_SELECT_MAX_KEYS), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    # first call on this device (when this test runs alone): looks up the built-in array and loads the kernels
    efm.beam_threshold_static(inputs[5][1].data_ptr(), cases[5][0], cases[5][1], out_static.data_ptr(), 0, stream)
    torch.cuda.synchronize()

    free_before, _ = torch.cuda.mem_get_info(dev)
    for i, ((n, cap, _, _), (k, d_k)) in enumerate(zip(cases, inputs)):   # back to back, no synchronisation in between
        efm.beam_threshold_static(d_k.data_ptr(), n, cap, out_static.data_ptr() + 8 * i, 0, stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(dev)[0] >= free_before   # no device memory was taken, by anyone, during the calls
    got = out_static.cpu().numpy().view(np.uint64)

    binding = []
    for i, ((n, cap, _, _), (k, d_k)) in enumerate(zip(cases, inputs)):
        want = threshold_by_definition(k, cap)
        assert int(got[i]) == want, f"case {i}: static {int(got[i]):#x} != definition {want:#x}"
        n_active = int((k < KEY_DONE).sum())
        if n_active > cap:   # the traversal runs its selection only when the beam binds
            efm.beam_threshold(d_k.data_ptr(), n, n_active, cap, scratch.data_ptr(), scratch.numel(), out_exist.data_ptr() + 8 * i,
                               0, stream)
            binding.append(i)
    exist = out_exist.cpu().numpy().view(np.uint64)
    assert len(binding) >= 5
    for i in binding:
        assert int(got[i]) == int(exist[i]), f"case {i}: static {int(got[i]):#x} != existing path {int(exist[i]):#x}"
    assert int(got[0]) == int(got[-1])                       # same input, other calls in between
    assert int(got[3]) == int(KEY_SENTINEL)                  # the beam did not bind
    # what the threshold means: exactly cap keys lie below it when the keys around it are distinct
    assert int((inputs[0][0] < got[0]).sum()) == cases[0][1]
    tied = inputs[2][0]                                       # sorted position cap lies inside a run of 45 972 equal keys
    assert int((tied == got[2]).sum()) > 40_000 and int((tied < got[2]).sum()) < cases[2][1]   # fewer are kept, never more
