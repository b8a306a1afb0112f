"""CPU oracle of the per-patch Godunov hydro/MHD update -- TEST INFRASTRUCTURE ONLY.

Importable from tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs, and from nowhere else.  See ``godunov_oracle.cpp`` for the method and
its pins; ``api.py`` is a ctypes binding; ``build.py`` compiles it with g++.
"""
