"""CPU oracle of the relaxation step (TEST INFRASTRUCTURE; see oracle/mro.c). Never imported by the product path."""
