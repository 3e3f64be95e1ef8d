"""Small case for compute-sanitizer (SURVEY aux row "sanitizers"); not collected by pytest.

    compute-sanitizer --tool memcheck|racecheck|initcheck python tests/sanitizer_case.py

40 x 30 x 20 three-phase image (a void and a fluid phase): the two-iteration kernel (DR_KERNEL 3, even and odd counts), the
one-sweep TMA kernel (DR_KERNEL 0), the split baseline (1), six load cases per launch (dr_solve_all), the averaging and export
kernels and dr_avg_stress_static.  Prints the averages so that a run under the sanitizer can be compared with a plain run."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def main():
    import torch
    from paper_2410_20441_b200 import binding
    rng = np.random.default_rng(40)
    ph = rng.integers(0, 3, size=(20, 30, 40))
    Kt = np.array([37.0, 0.0, 2.2]); Gt = np.array([44.0, 0.0, 0.0])
    K = torch.from_numpy(np.ascontiguousarray(Kt[ph])).cuda()
    G = torch.from_numpy(np.ascontiguousarray(Gt[ph])).cuda()
    out = []
    for kernel, niter in ((3, 6), (3, 5), (0, 3), (1, 2)):
        s = binding.Solver(K, G, kernel=kernel)
        s.step(4, 1e-4, niter)
        assert s.active_kernel() == kernel
        out.append(s.avg_stress())
        fields = [s.get_field(f) for f in range(3, 9)]
        st = binding.avg_stress_static(fields).cpu().numpy()
        assert np.max(np.abs(st - out[-1])) <= 1e-10 * np.max(np.abs(out[-1]))
        s.close()
    b = binding.Solver(K, G, six=True, ncheck=4)
    C, log = b.solve_all_batched(1e-4, 1e-30, 10)
    assert b.active_kernel() == 3 and all(l[1] == 10 for l in log)
    torch.cuda.synchronize()
    print("sanitizer case ok:", " ".join("%.12e" % v for v in out[0]), "C33 %.12e" % C[2, 2])


if __name__ == "__main__":
    main()
