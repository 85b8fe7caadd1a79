"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the method (no stencil, no potential sum, no
mask, no packet evaluation): it only produces *inputs* -- grid sizes, boundary
flags, atom lists, packet parameters, detector parameters -- for the five
configurations of BASELINE.json.  Both `oracle/` and `paper_2401_07416_b200/`
consume these inputs; neither imports the other.

The inputs stand in for the paper's Cu(111) and Au(111)/C6-SAM workloads
(section 2.3), whose DFT potentials and structure files are not
available; see DESIGN.md "Input recipe".
"""
from .configs import (Workload, make_config, fcc111_slab, molecule_template, CONFIG_NAMES,
                      random_state, random_potential, shard_for_rank, PERIODIC, DIRICHLET, PaperMesh, paper_mesh)

__all__ = ["Workload", "make_config", "fcc111_slab", "molecule_template", "CONFIG_NAMES",
           "random_state", "random_potential", "shard_for_rank", "PERIODIC", "DIRICHLET", "PaperMesh", "paper_mesh"]
