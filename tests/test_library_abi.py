"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol that
include/pyjac_b200.h declares, validates descriptions before touching CUDA, and fails loudly
(PYJAC_ECUDA, never a CPU fallback) when no device is usable."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1605_03262_b200 import binding, build, synth
from paper_1605_03262_b200.mechanism import FALLOFF, PLOG, THIRD_BODY, MechanismBuilder

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def declared_symbols(header):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pyjac_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    """Every function include/pyjac_b200.h declares is exported by the product library, and nothing of
    the bench / test helper interface is; the helper library exports exactly its own header."""
    names = declared_symbols("pyjac_b200.h")
    assert set(names) == set(binding.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n
    tools = binding.load_tools()
    tnames = declared_symbols("pyjac_b200_tools.h")
    assert set(tnames) == set(binding.TOOLS_EXPORTS)
    for n in tnames:
        assert hasattr(tools, n), n
        assert not hasattr(lib, n), n


def test_product_library_reads_no_environment(lib):
    """no runtime flags beyond the call arguments -- none of the product's own object
    files references getenv (launch shapes are an explicit argument of pyjac_mech_create_shaped; the CUDA
    runtime linked into the .so reads its own variables, which is not ours to change)."""
    import glob
    import subprocess
    objs = [o for o in glob.glob(os.path.join(os.path.dirname(binding.LIB_PATH), "build", "*.o"))
            if not o.endswith("tools.o")]
    assert len(objs) >= 4
    for o in objs:
        out = subprocess.run(["nm", "--undefined-only", o], capture_output=True, text=True).stdout
        assert "getenv" not in out, o


def test_strerror(lib):
    for code in (0, -1, -2, -3, -4, -99):
        assert lib.pyjac_strerror(code)
    assert b"success" in lib.pyjac_strerror(0)


def _create(lib, mech):
    d, keep = binding.mech_desc(mech)
    h = C.c_void_p()
    rc = lib.pyjac_mech_create(C.byref(d), 0, C.byref(h))
    if rc == 0:
        lib.pyjac_mech_destroy(h)
    return rc


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def test_create_fails_loudly_without_a_device(lib):
    """No GPU here: a valid description must give PYJAC_ECUDA, not a silent fallback."""
    rc = _create(lib, synth.make_mechanism(0))
    assert rc == (binding.PYJAC_OK if _has_gpu() else binding.PYJAC_ECUDA)


def test_null_and_degenerate_arguments(lib):
    assert lib.pyjac_mech_create(None, 0, None) == binding.PYJAC_EINVAL
    h = C.c_void_p()
    assert lib.pyjac_mech_create(None, 0, C.byref(h)) == binding.PYJAC_EINVAL
    assert lib.pyjac_mech_destroy(None) == binding.PYJAC_OK
    assert lib.pyjac_mech_sizes(None, None, None) == binding.PYJAC_EINVAL
    assert lib.pyjac_eval_jacobian(None, 1, None, None, None, 1, None, None) == binding.PYJAC_EINVAL
    assert lib.pyjac_eval_jacobian_host(None, 1, None, None, None, 1, None, 0) == binding.PYJAC_EINVAL
    assert lib.pyjac_kernel_launches() >= 0


def _base():
    m = synth.make_tiny_mechanism(0)
    return m


@pytest.mark.parametrize("what", ["spec_range", "nu_range", "four_species", "neg_A", "plog_order",
                                  "cheb_lim", "eff_range", "rxn_type", "repeat_species", "tb_range"])
def test_validation_rejects_bad_descriptions(lib, what):
    """pyjac_mech_create validates on the host before any CUDA call (PYJAC_EINVAL)."""
    m = _base()
    if what == "spec_range":
        m.reac_spec = m.reac_spec.copy(); m.reac_spec[0] = m.n_species
    elif what == "nu_range":
        m.prod_nu = m.prod_nu.copy(); m.prod_nu[0] = 4
    elif what == "four_species":
        b = MechanismBuilder(m.species_names, m.element_names, m.composition, m.mol_wt, m.nasa_lo,
                             m.nasa_hi, m.t_mid)
        b.add([(0, 1), (1, 1), (2, 1), (3, 1)], [(4, 1)], (1.0, 0.0, 0.0))
        m = b.build()
    elif what == "neg_A":
        i = int(np.where(m.rxn_type == 0)[0][0])
        m.arr_hi = m.arr_hi.copy(); m.arr_hi[i, 0] = -1.0
    elif what == "plog_order":
        i = int(np.where(m.rxn_type == PLOG)[0][0])
        m.plog_p = m.plog_p.copy(); b = m.plog_ptr[i]; m.plog_p[b + 1] = m.plog_p[b]
    elif what == "cheb_lim":
        i = int(np.where(m.rxn_type == 5)[0][0])
        m.cheb_lim = m.cheb_lim.copy(); m.cheb_lim[i, 1] = m.cheb_lim[i, 0]
    elif what == "eff_range":
        m.eff_spec = m.eff_spec.copy(); m.eff_spec[0] = -1
    elif what == "rxn_type":
        m.rxn_type = m.rxn_type.copy(); m.rxn_type[0] = 6
    elif what == "repeat_species":
        b = MechanismBuilder(m.species_names, m.element_names, m.composition, m.mol_wt, m.nasa_lo,
                             m.nasa_hi, m.t_mid)
        b.add([(0, 1), (0, 1)], [(4, 1)], (1.0, 0.0, 0.0))
        m = b.build()
    elif what == "tb_range":
        i = int(np.where(m.rxn_type == THIRD_BODY)[0][0])
        m.tb_species = m.tb_species.copy(); m.tb_species[i] = m.n_species
    assert _create(lib, m) == binding.PYJAC_EINVAL
    assert len(lib.pyjac_mech_create_error()) > 8          # the broken rule is named, not just the code


def test_binding_refuses_cpu_tensors():
    """The product path never computes on the CPU: the binding rejects non-CUDA tensors."""
    import torch
    pj = binding.PyJac.__new__(binding.PyJac)
    pj.ns, pj.nr = 3, 1
    with pytest.raises(TypeError):
        pj._dev_inputs(torch.zeros(2, dtype=torch.float64), torch.zeros(2, dtype=torch.float64),
                       torch.zeros(2, 3, dtype=torch.float64))


@pytest.mark.parametrize("shape", [
    None, dict(states_per_cta=1), dict(states_per_cta=2, ctas_per_sm=3, threads=160), dict(states_per_cta=6),
    dict(states_per_cta=4, ctas_per_sm=1), dict(states_per_cta=1, threads=64), dict(list_cap=6), dict(list_cap=64),
    dict(cell_cap=1), dict(cell_cap=2, rows_per_lane=1), dict(layout=2), dict(p1_states=1), dict(p1_states=3 + 16 * 1),
    dict(states_per_cta=2, threads=512, ctas_per_sm=1, stage_tables=1),
])
def test_pack_self_check_over_launch_shapes(shape):
    """pyjac_tools_pack_stats packs exactly as pyjac_mech_create_shaped does, including the self-check of
    everything the kernels read without bounds checks (whole rows of chunks, table blocks, entry offsets);
    it must hold for every configuration and every launch shape."""
    for cfg in (0, 1, 2, 3):
        try:
            st = binding.pack_stats(synth.make_mechanism(cfg), shape)
        except binding.PyJacError as e:
            # a forced shape that does not fit the shared memory of one CTA is refused, loudly
            assert e.code == binding.PYJAC_ELIMIT and shape is not None and cfg >= 1
            continue
        assert st["chunks"] > 0 and st["states_per_cta"] >= 1 and st["smem_bytes_per_cta"] <= 227 * 1024
        assert st["threads"] % 32 == 0 and st["threads"] >= 32 * st["states_per_cta"]
    for seed in range(4):
        binding.pack_stats(synth.make_tiny_mechanism(seed), shape)


def test_layout_search_lowers_the_modelled_bank_conflicts():
    """mech_pack.cu: the layout search of the per-reaction terms (indices traded within a store wavefront against
    the gather groups) and the exact edge colouring of the gather steps.  Host-only model (shared-memory wavefronts
    beyond one per lane group and step): the streaming phase must be nearly conflict-free and the capacity excess of
    the gather groups must drop by more than half; with layout = 2 (allocation order) the excess is not computed."""
    for cfg in (1, 2, 3):
        m = synth.make_mechanism(cfg)
        on, off = binding.pack_stats(m), binding.pack_stats(m, dict(layout=2))
        assert on["layout_excess_before"] > 0 and 2 * on["layout_excess_after"] < on["layout_excess_before"]
        assert off["layout_excess_before"] == 0 and off["layout_excess_after"] == 0
        assert on["b_conflict_wf"] < off["b_conflict_wf"] and on["a_conflict_wf"] < off["a_conflict_wf"]
        assert on["b_conflict_wf"] <= 0.02 * on["b_steps"] * 2
        for k in ("e_elements", "cell_entries", "a_steps", "b_steps", "smem_bytes_per_cta"):
            assert on[k] == off[k]                      # a permutation: nothing else changes


def test_gather_probe_tables_cover_every_cell_list():
    """Helper library, host half of the gather timing prototype (profiles/r3_gather_probe.md): its chunk tables are built
    before any CUDA call, so without a GPU the call ends with PYJAC_ECUDA but has already reported what it built -- every
    entry of every non-empty cell list (the same counts pyjac_tools_pack_stats reports), dealt into chunks of 32 cells
    of nearly equal length (little padding), and a shared-memory size that grows with S and the tile sets."""
    tools = binding.load_tools()
    for cfg in (0, 1, 2):
        m = synth.make_mechanism(cfg)
        d, keep = binding.mech_desc(m)
        ld = m.n_species + 1
        st0 = binding.pack_stats(m)
        seen = []
        out_ptr, out_keep = C.c_void_p(16), None                  # never dereferenced without a device
        if _has_gpu():                                            # with one the probe really runs: give it real memory
            import torch
            out_keep = torch.empty(100 * ld * ld, dtype=torch.float64, device="cuda")
            out_ptr = C.c_void_p(out_keep.data_ptr())
        for S, nbuf in ((1, 1), (3, 2)):
            exp = np.full(ld * ld, np.nan)
            stats = (C.c_int64 * 8)()
            a, b = C.c_float(), C.c_float()
            rc = tools.pyjac_tools_gather_probe(C.byref(d), S, 256, 1, nbuf, 100, out_ptr, exp.ctypes.data_as(binding._pd),
                                                stats, 1, C.byref(a), C.byref(b), None)
            assert rc in ((binding.PYJAC_OK, binding.PYJAC_ELIMIT) if _has_gpu() else (binding.PYJAC_ECUDA,))
            entries, padded, chunks, n_e, smem, nonempty, cells, _ = list(stats)
            assert cells == ld * ld and nonempty == st0["cells"] and entries == st0["cell_entries"] and n_e == st0["e_elements"]
            assert chunks == (nonempty + 31) // 32 and entries <= padded <= 1.25 * entries + 32 * 16
            assert smem == (((n_e * S + 15) // 16 * 16) + nbuf * S * cells) * 8
            assert np.all(np.isfinite(exp))                       # the expected tile was filled for every cell
            seen.append(exp.copy())
        assert np.array_equal(seen[0], seen[1])                   # it does not depend on the launch shape
    assert tools.pyjac_tools_gather_probe(None, 1, 256, 1, 1, 1, None, None, None, 1, None, None, None) == binding.PYJAC_EINVAL


def test_launch_shape_validation():
    m = synth.make_mechanism(0)
    for bad in (dict(states_per_cta=5), dict(threads=100), dict(threads=1024), dict(ctas_per_sm=9),
                dict(cell_cap=4), dict(rows_per_lane=3), dict(states_per_cta=-1),
                # explicit values are never adjusted: too few threads for the interleaved states,
                # fewer than two warps, a negative field
                dict(states_per_cta=3, threads=64), dict(threads=32), dict(p1_states=-1), dict(threads=-32)):
        with pytest.raises(binding.PyJacError) as e:
            binding.pack_stats(m, bad)
        assert e.value.code == binding.PYJAC_EINVAL
    with pytest.raises(binding.PyJacError) as e:       # two rows per lane need an even leading dimension: 360 species is even
        binding.pack_stats(synth.make_mechanism(3), dict(rows_per_lane=2))
    assert e.value.code == binding.PYJAC_EINVAL
    assert binding.pack_stats(m, dict(rows_per_lane=2, threads=64, states_per_cta=2))["threads"] == 64
    with pytest.raises(ValueError):
        binding.launch_shape(dict(no_such_field=1))


def test_binding_validates_outputs():
    """Outputs are written in place and never copied or converted: a wrong dtype, a non-contiguous view or a
    buffer that is too small is an error, not a silent temporary."""
    pj = binding.PyJac.__new__(binding.PyJac)
    pj.ns, pj.nr, pj.device = 3, 1, 0
    for bad in (np.zeros((4, 16), dtype=np.float32), np.zeros((4, 32))[:, ::2], np.zeros((4, 15)), [[0.0] * 16] * 4):
        with pytest.raises(ValueError):
            pj._host_out(bad, 4 * 16)
    assert pj._host_out(np.zeros((4, 16)), 4 * 16) != 0
