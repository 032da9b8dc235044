"""Test and benchmark harness (not part of the product library): the seeded synthetic workload
generators, the host stand-in for the engine's prefix cache they use to build cache inputs, and the
random-sector gather probe bench.py measures its ceiling with.  Holds none of the method's arithmetic."""
