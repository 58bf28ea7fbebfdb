"""CPU oracle for the coupled-oscillator RK4 hot path (TEST INFRASTRUCTURE).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this package.  It never imports the CUDA
package and shares no code with it.
"""
