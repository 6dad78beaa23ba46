"""TEST INFRASTRUCTURE: the cases tests/test_simt_kernels.py runs in a child process against a sanitizer build of the
emulation: `python san_cases.py` = -fsanitize=address,undefined (libasan preloaded), `python san_cases.py tsan` =
ThreadSanitizer on the kernels (libtsan preloaded; one TSan fibre per CUDA thread, happens-before only where CUDA gives
it).  `python san_cases.py overrun` is the self-test that must die with an AddressSanitizer report."""
import ctypes as C
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path[:0] = [os.path.dirname(os.path.dirname(HERE)), os.path.dirname(HERE), HERE]

from harness import Emu, load  # noqa: E402


def main():
    if sys.argv[1:] == ["overrun"]:
        L = load(sanitize=True)
        L.simt_selftest_overrun.argtypes = [C.c_void_p, C.c_size_t]
        p = L.simt_alloc(4096)
        L.simt_selftest_overrun(p, 4096)
        print("SIMT-SAN the overrun went unnoticed")
        return
    import test_gpu_parity as gp
    import test_gpu_readouts as gr
    import test_gpu_traces as gt
    import test_zz_gpu_global_tables as gz

    from workloads import configs

    def w3_shell_and_nucleus(e):       # membrane crossings, no-flux walls, expression channels
        gp.run_both(e, configs.w3(scale=0.004, n_steps=60, cell_size=1024), 60, chunks=2)

    mode = "tsan" if sys.argv[1:] == ["tsan"] else True
    emu = Emu(sanitize=mode)
    def random_models(e):              # 30 random models: every shape, channel kind, homodimers, replicas, crowded volumes
        from paper_2606_14603_b200.binding import check_config
        from random_models import fuzz_parity

        assert fuzz_parity(e, range(200, 230), check_config, gp.oracle_cls(), gp.assert_same) >= 25

    cases = [gp.test_tiny_dense_cube_many_events, gp.test_channel_kinds_and_priority, gp.test_crowded_single_cell,
             gt.test_homodimer_parity, gp.test_empty_population_and_mid_run_seeding, gp.test_errors,
             gt.test_load_agents_rejects_bad_positions_and_duplicate_ids, gr.test_picture_parity_nucleus_and_cytoplasm,
             w3_shell_and_nucleus, gz.body_large_gaussian_tables, gz.body_maximum_table_sizes,
             gz.body_degenerate_populations, random_models]
    import time

    if mode == "tsan":                 # the race check proper: the kernels that share queues, tiles and counters
        def random_models_few(e):
            from paper_2606_14603_b200.binding import check_config
            from random_models import fuzz_parity

            assert fuzz_parity(e, range(200, 212), check_config, gp.oracle_cls(), gp.assert_same) >= 9

        cases = [gp.test_tiny_dense_cube_many_events, gp.test_channel_kinds_and_priority, gp.test_crowded_single_cell,
                 gt.test_homodimer_parity, gp.test_errors, w3_shell_and_nucleus, gz.body_maximum_table_sizes,
                 random_models_few]
    for c in cases:
        t0 = time.time()
        c(emu)
        print(f"SIMT-SAN case ok: {c.__name__} ({time.time() - t0:.1f} s)", flush=True)
    print(f"SIMT-SAN OK {len(cases)} cases, {load(mode).simt_launches()} kernel launches", flush=True)


if __name__ == "__main__":
    main()
